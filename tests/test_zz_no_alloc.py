"""fk_conv_hadronic_static (include/fkconv.h): the forward convolution, Eq. (1), for callers that cannot
allocate device memory.  Its scratch is a file-scope static device array of FK_STATIC_SCRATCH_BYTES inside the library.

Collected last on purpose (the suite runs with `pytest -x`).  Passes alone in a fresh process and after the other tests:
nothing here depends on what an earlier call left in the shared array, and the second call of every pair checks exactly
that (other sizes, another code path, stale contents from the first call).
"""
import numpy as np
import pytest

from oracle import fk_oracle as O
from paper_1909_10547_b200 import synth
from tests._parity import TOL64, rel_err, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def K():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    from paper_1909_10547_b200 import fkconv
    return fkconv


def _both(K, case):
    """(static-scratch result, existing stateless path's result, oracle, scale) of one case."""
    import torch
    fk_d, f_d = to_dev(case.fk), to_dev(case.f)
    sig = torch.full((case.N, case.f.shape[0]), float("nan"), dtype=torch.float64, device="cuda")   # caller's output buffer
    K.fk_conv_hadronic_static(fk_d, case.pairs, f_d, sig)
    want = K.fk_conv_hadronic(fk_d, case.pairs, f_d)
    torch.cuda.synchronize()
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    return sig.cpu().numpy(), want.cpu().numpy(), ref, scale


def test_static_scratch_forward_two_calls_in_a_row(K):
    """Two calls in a row on different problems: (1) several k-blocks and datapoint ranges at R = 3 (level-1 partials in
    the array, two-level reduction); (2) a smaller table at R = 2 whose partials land on top of the first call's.  Each
    against the existing path (fk_conv_hadronic, stream-ordered scratch) within the fp64 bar, and against the oracle."""
    first = synth.hadronic_case(31, 70, 30, 17, 3, sub=1)     # K = 15 300: 30 k-blocks
    second = synth.hadronic_case(31, 33, 20, 9, 2, sub=2)     # K = 3 600: 8 k-blocks, stale partials beyond them
    for case in (first, second, first):
        got, want, ref, scale = _both(K, case)
        assert np.isfinite(got).all()
        assert rel_err(got, want, scale) <= TOL64
        assert rel_err(got, ref, scale) <= TOL64


def test_static_scratch_dense_path_after_column_path(K):
    """R = 40 takes the FP64 tensor-core contraction (replica-innermost f, split-K partials, k codes: all in the array);
    then R = 1 on the same table reuses the same bytes as level-1 partials."""
    dense = synth.hadronic_case(32, 150, 20, 12, 40, sub=3)
    one = synth.hadronic_case(32, 150, 20, 12, 1, sub=3)
    for case in (dense, one):
        got, want, ref, scale = _both(K, case)
        assert rel_err(got, want, scale) <= TOL64 and rel_err(got, ref, scale) <= TOL64


def test_static_scratch_single_k_block_needs_no_scratch(K):
    case = synth.hadronic_case(33, 9, 6, 5, 2, sub=4)         # K = 180: one k-block, sigma written directly
    got, want, ref, scale = _both(K, case)
    assert rel_err(got, want, scale) <= TOL64 and rel_err(got, ref, scale) <= TOL64


def test_static_scratch_rejects_sizes_beyond_the_array(K):
    """A problem whose level-1 partials exceed FK_STATIC_SCRATCH_BYTES: FK_ERR_UNSUPPORTED, a message that names the need
    and the limit, nothing launched (the output keeps its contents).  The table itself is never read: a small buffer
    stands in for it, so the test needs no memory."""
    import torch
    N, nx, C, R, nfl = 4096, 64, 128, 4, 14            # 4096 x 1024 k-blocks x 4 replicas x 8 B = 128 MiB
    fk_stub = torch.zeros((1,), dtype=torch.float64, device="cuda")
    f = torch.zeros((R, nfl, nx), dtype=torch.float64, device="cuda")
    sig = torch.full((N, R), 7.0, dtype=torch.float64, device="cuda")
    pairs = np.zeros((C, 2), dtype=np.int32)
    rc = K.lib.fk_conv_hadronic_static(fk_stub.data_ptr(), pairs.ctypes.data, f.data_ptr(), sig.data_ptr(), N, nx, nfl, C, R, 0)
    assert rc == K.FK_ERR_UNSUPPORTED
    msg = K.lib.fk_last_error_string().decode()
    assert "FK_STATIC_SCRATCH_BYTES" in msg and str(K.FK_STATIC_SCRATCH_BYTES) in msg
    torch.cuda.synchronize()
    assert bool((sig == 7.0).all())
    # the next call still works
    case = synth.hadronic_case(31, 33, 20, 9, 2, sub=2)
    got, want, ref, scale = _both(K, case)
    assert rel_err(got, want, scale) <= TOL64
