"""CPU oracle for the FK convolution - TEST INFRASTRUCTURE (see fk_oracle.c header).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference may import this."""
