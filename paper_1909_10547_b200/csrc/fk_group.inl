// fk_group.inl -- ragged grouped launch; included at the end of fk_api.cu.
// A global fit convolves many tables of different (N, nx, C) every iteration.  The
// host builds, once, static work lists of (table, k-block, datapoint range) CTAs; a forward pass is
// then ONE column-kernel launch (+ one level-2 reduce) over all tables, a VJP pass one column-sum
// launch + one gather launch; the hardware CTA scheduler balances the ragged list.  Every partial has
// a fixed slot and every sum a fixed order, so results are bitwise repeatable.

struct fk_group {
    HandleSync sync;
    std::vector<fk_table*> tables;
    std::vector<fk::TableDesc> descs;  // host copies with the concatenation offsets filled in
    int T = 0, dtype = FK_F64;
    bool all_vec = true;
    long long rows_total = 0, ai_total = 0, f_total1 = 0, part_total1 = 0, G_total1 = 0, elems_total = 0;
    fk::TableDesc* d_descs = nullptr;
    int* d_row_prefix = nullptr;
    int* d_ai_prefix = nullptr;
    fk::ColSeg* d_fsegs = nullptr;  // forward CTAs: (table, k-block, datapoint range)
    int nfsegs = 0;
    fk::ColSeg* d_csegs = nullptr;  // VJP stage-1 CTAs
    int ncsegs = 0;
    // R >> 1 contraction (fk_gemm.cuh): items {table, datapoint tile, K range} / {table, 128-k tile}
    bool gemm_ok = false;
    fk::ColSeg* d_gitems = nullptr;
    int ngitems = 0;
    fk::ColSeg* d_vitems = nullptr;
    int nvitems = 0;
    long long gp_rows = 0, K_total = 0, cx_total = 0;
    bool ws_all = true;             // every table can take the warp-specialised forward contraction (fk_gemm_ws.cuh)
    bool jp_all = true;             // no table pads its x-rows (jp == nx): the forward contraction walks k with nx
    int nx_max = 0;
    fk::ColSeg* d_witems = nullptr; // its items: {table, first datapoint, K range of the item, k sub-splits}
    int nwitems = 0;
    bool foldk_all = true;          // every table can take the small-R single-pass fold (fk_vjp_foldk_kernel)
    fk::ColSeg* d_kitems = nullptr; // its CTAs: {table, channel}
    int nkitems = 0;
    bool wsv_all = true;            // every table can take the persistent warp-specialised VJP contraction
    bool fold_all = true;           // every table can take the single-pass VJP fold (fk_vjp_fold.cuh)
    int fold_nchunk = 1;
    fk::ColSeg* d_foitems = nullptr;  // fold CTAs: {table, channel, x-row chunk}
    int nfoitems = 0;
    // fp32 variant at R >> 1: tcgen05 contraction over the group (fk_tc32.cu): items {table, first datapoint, range of (c, i) rows}
    bool tc_all = false;
    fk::ColSeg* d_tcitems = nullptr;
    int ntcitems = 0;
    long long tc_gp_rows = 0;
    // forward + VJP from one read of FK (fk_fused_column_kernel, GROUPED): the datapoint ranges of the fused CTAs
    // (<= 64 rows) are also the slices of the column sums, so the group keeps a second set of descriptors
    bool fused_all = true;
    fk::TableDesc* d_descs_fused = nullptr;
    fk::ColSeg* d_usegs = nullptr;
    int nusegs = 0;
    long long G_total1_fused = 0;
    int* d_l2cnt = nullptr;   // tickets of the forward kernel's in-kernel level-2 reduction, one per (table, datapoint range)
    long long cnt_total = 0;
    double* scratch = nullptr;
    size_t scratch_elems = 0;
    int last_launches = 0;
};

namespace {

int group_scratch(fk_group* g, size_t elems, cudaStream_t s = nullptr) {
    if (elems <= g->scratch_elems) return FK_OK;
    if (stream_capturing(s))
        return fail(FK_ERR_UNSUPPORTED, "the group's scratch must grow to %zu doubles, which cannot happen during stream capture: "
                                        "give R_hint at create or make one call outside the capture first", elems);
    if (g->scratch) cudaFree(g->scratch);
    g->scratch = nullptr;
    g->scratch_elems = 0;
    FK_CUDA(cudaMalloc((void**)&g->scratch, elems * sizeof(double)));
    g->scratch_elems = elems;
    return FK_OK;
}

bool group_gemm_wanted(const fk_group* g, int R) {
    return g->gemm_ok && g->dtype == FK_F64 && R >= (opt(FK_OPT_GEMM_MIN_R) > 0 ? opt(FK_OPT_GEMM_MIN_R) : g->ws_all ? 5 : 13);
}

// groups of fp32-STORED tables at R >> 1 (fk_api.cu, vjp32_wanted / fwd32_wanted): the FP64 contractions over the tables as stored
bool group_vjp32_wanted(const fk_group* g, int R) {
    return g->dtype != FK_F64 && g->wsv_all && opt(FK_OPT_WARP_SPEC) &&
           R >= (opt(FK_OPT_GEMM_MIN_R) > 0 ? opt(FK_OPT_GEMM_MIN_R) : VJP32_DEFAULT_MIN_R);
}
bool group_fwd32_wanted(const fk_group* g, int R) {
    return g->dtype == FK_F32S64 && g->ws_all && g->jp_all && opt(FK_OPT_WARP_SPEC) &&
           fk::ws_smem_bytes(g->nx_max, fk::gemm_rp(R)) <= MAX_DYN_SMEM &&
           R >= (opt(FK_OPT_GEMM_MIN_R) > 0 ? opt(FK_OPT_GEMM_MIN_R) : FWD32_DEFAULT_MIN_R);
}

size_t group_tc32_scratch_need(const fk_group* g, int R);
bool group_tc32_wanted(const fk_group* g, int R);

size_t group_scratch_need(const fk_group* g, int R) {
    const size_t RP = fk::gemm_rp(R);
    const size_t gemm_fwd = ((size_t)g->ai_total + (size_t)g->gp_rows) * RP,
                 gemm_vjp = ((size_t)g->ai_total + (size_t)g->rows_total + (size_t)g->K_total + (size_t)g->cx_total * (fk::FOLD_JQ + g->fold_nchunk)) * RP;
    if (group_gemm_wanted(g, R)) return std::max(gemm_fwd, gemm_vjp);
    size_t need = std::max<size_t>((size_t)g->part_total1, (size_t)g->G_total1 + (1 + FOLDK_MAX_CHUNKS) * (size_t)g->cx_total) * R;
    if (group_tc32_wanted(g, R)) need = std::max(need, group_tc32_scratch_need(g, R));
    if (group_fwd32_wanted(g, R)) need = std::max(need, gemm_fwd);
    if (group_vjp32_wanted(g, R)) need = std::max(need, gemm_vjp);
    return need;
}

// ---- fp32 variant at R >> 1 over a group: one tcgen05 launch per pass of <= 128 replicas ----
bool group_tc32_wanted(const fk_group* g, int R) {
    return g->tc_all && g->dtype == FK_F32 && opt(FK_OPT_TC32) && R >= (opt(FK_OPT_TC32_MIN_R) > 0 ? opt(FK_OPT_TC32_MIN_R) : TC32_DEFAULT_MIN_R);
}
// scratch in doubles: fT32 [slots of the group][RPmax] floats + level-1 partials [tc_gp_rows][RPmax] floats
size_t group_tc32_scratch_need(const fk_group* g, int R) {
    const size_t RP = fk::tc_rp(R);
    return (((size_t)g->ai_total * RP + 31) / 32 * 32 + (size_t)g->tc_gp_rows * RP + 1) / 2 + 64;
}
int group_conv_tc32(fk_group* g, const float* f_cat, float* sigma_cat, int R, cudaStream_t s) {
    const int RPmax = fk::tc_rp(R);
    float* fT = reinterpret_cast<float*>(g->scratch);
    float* gpart = fT + ((size_t)g->ai_total * RPmax + 31) / 32 * 32;   // 128-byte aligned
    int nl = 0;
    for (int r0 = 0; r0 < R; r0 += fk::TC_MAX_RP) {
        fk::Tc32Params p;
        memset(&p, 0, sizeof p);
        p.fT = fT;
        p.gpart = gpart;
        p.RP = fk::tc_rp(R - r0);
        p.descs = g->d_descs;
        p.items = g->d_tcitems;
        const long long tf = g->ai_total * p.RP;
        FK_TIMED("fk_transpose_f_grouped", s) fk::fk_transpose_f_grouped_kernel<float, float><<<(int)std::min<long long>(4096, (tf + 255) / 256), 256, 0, s>>>(
            f_cat, fT, g->d_ai_prefix, g->T, g->ai_total, R, r0, p.RP);
        cudaError_t e = cudaSuccess;
        FK_TIMED("fk_tc32_fwd", s) e = fk::tc32_fwd_launch(p, g->ntcitems, true, false, s);
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "grouped tcgen05 forward launch failed: %s", cudaGetErrorString(e));
        const long long outs = g->rows_total * p.RP;
        FK_TIMED("fk_gemm_reduce_grouped", s) launch_pdl(fk::fk_gemm_reduce_grouped_kernel<float, float, true>, (int)std::min<long long>(8192, (outs + 255) / 256), 256, 0, s,
                                                         gpart, sigma_cat, g->d_descs, g->d_row_prefix, g->T, g->rows_total, R, r0, p.RP);
        e = cudaGetLastError();
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "grouped tcgen05 reduce launch failed: %s", cudaGetErrorString(e));
        nl += 3;
    }
    g->last_launches = nl;
    return FK_OK;
}

bool group_fused_wanted(const fk_group* g, int R) {
    return g->fused_all && !group_gemm_wanted(g, R) && R <= 4 && opt(FK_OPT_FUSED);
}
// part [rows][R][nchunks] | G [fused splits][R][K] | fold partials
size_t group_fused_scratch_need(const fk_group* g, int R) {
    return ((size_t)g->part_total1 + (size_t)g->G_total1_fused + (1 + FOLDK_MAX_CHUNKS) * (size_t)g->cx_total) * R;
}

// TS = storage type of the tables (float: FK_F32S64 groups, warp-specialised kernel only)
template <typename TS = double>
int group_conv_gemm(fk_group* g, const double* f_cat, double* sigma_cat, int R, cudaStream_t s) {
    const int RPmax = fk::gemm_rp(R);
    double* fT = g->scratch;
    double* gpart = fT + (size_t)g->ai_total * RPmax;
    if (!(ensure_dyn_smem(fk::fk_gemm_fwd_kernel<2, true>, fk::GEMM_SMEM_BYTES) && ensure_dyn_smem(fk::fk_gemm_fwd_kernel<1, true>, fk::GEMM_SMEM_BYTES)))
        return fail(FK_ERR_CUDA, "grouped gemm: cannot reserve %d bytes of shared memory", fk::GEMM_SMEM_BYTES);
    int nl = 0;
    for (int r0 = 0; r0 < R; r0 += fk::GEMM_BN) {
        fk::GemmFwdParams p;
        memset(&p, 0, sizeof p);
        p.fT = fT;
        p.gpart = gpart;
        p.RP = fk::gemm_rp(R - r0);
        p.nfrag = p.RP / 8;
        p.nfw = (p.nfrag + 1) / 2;
        p.descs = g->d_descs;
        p.items = g->d_gitems;
        const long long tf = g->ai_total * p.RP;
        FK_TIMED("fk_transpose_f_grouped", s) fk::fk_transpose_f_grouped_kernel<double><<<(int)std::min<long long>(4096, (tf + 255) / 256), 256, 0, s>>>(
            f_cat, fT, g->d_ai_prefix, g->T, g->ai_total, R, r0, p.RP);
        const size_t ws_smem = fk::ws_smem_bytes(g->nx_max, p.RP);
        if (g->ws_all && opt(FK_OPT_WARP_SPEC) && ws_smem <= MAX_DYN_SMEM) {
            fk::WsFwdParams w;
            memset(&w, 0, sizeof w);
            w.fT = fT;
            w.gpart = gpart;
            w.RP = p.RP;
            w.descs = g->d_descs;
            w.items = g->d_witems;
            if (!ws_launch<true, TS>(w, g->nwitems, ws_smem, s))
                return fail(FK_ERR_CUDA, "grouped gemm: cannot reserve %zu bytes of shared memory", MAX_DYN_SMEM);
        } else if (!std::is_same<TS, double>::value) return fail(FK_ERR_UNSUPPORTED, "grouped gemm: fp32-stored tables without the packed bulk-copy layout");
        else if (g->all_vec) FK_TIMED("fk_gemm_fwd", s) fk::fk_gemm_fwd_kernel<2, true><<<g->ngitems, fk::GEMM_THREADS, fk::GEMM_SMEM_BYTES, s>>>(p);
        else FK_TIMED("fk_gemm_fwd", s) fk::fk_gemm_fwd_kernel<1, true><<<g->ngitems, fk::GEMM_THREADS, fk::GEMM_SMEM_BYTES, s>>>(p);
        const long long outs = g->rows_total * p.RP;
        FK_TIMED("fk_gemm_reduce_grouped", s) fk::fk_gemm_reduce_grouped_kernel<double><<<(int)std::min<long long>(8192, (outs + 255) / 256), 256, 0, s>>>(
            gpart, sigma_cat, g->d_descs, g->d_row_prefix, g->T, g->rows_total, R, r0, p.RP);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "grouped gemm forward launch failed: %s", cudaGetErrorString(e));
        nl += 3;
    }
    g->last_launches = nl;
    return FK_OK;
}

// T = type of f, g, df; TS = storage type of the tables (fk_api.cu, run_vjp_gemm)
template <typename T = double, typename TS = double>
int group_vjp_gemm(fk_group* g, const T* f_cat, const T* g_cat, T* df_cat, int R, cudaStream_t s) {
    if (!std::is_same<TS, double>::value && !g->wsv_all) return fail(FK_ERR_UNSUPPORTED, "grouped gemm vjp: fp32-stored tables without 16-byte aligned rows");
    const int RPmax = fk::gemm_rp8(R);
    double* fT = g->scratch;
    double* gP = fT + (size_t)g->ai_total * RPmax;
    double* G = gP + (size_t)g->rows_total * RPmax;
    if (!(ensure_dyn_smem(fk::fk_gemm_vjp_kernel<2, true>, fk::GEMMV_SMEM_BYTES) && ensure_dyn_smem(fk::fk_gemm_vjp_kernel<1, true>, fk::GEMMV_SMEM_BYTES)))
        return fail(FK_ERR_CUDA, "grouped gemm vjp: cannot reserve %d bytes of shared memory", fk::GEMMV_SMEM_BYTES);
    int nl = 0;
    for (int r0 = 0; r0 < R; r0 += fk::GEMM_BN) {
        const int RP = fk::gemm_rp8(R - r0);
        const long long tf = g->ai_total * RP, tg = g->rows_total * RP;
        FK_TIMED("fk_transpose_f_grouped", s) fk::fk_transpose_f_grouped_kernel<T, double><<<(int)std::min<long long>(4096, (tf + 255) / 256), 256, 0, s>>>(
            f_cat, fT, g->d_ai_prefix, g->T, g->ai_total, R, r0, RP);
        // g_cat is [global row][R]: the single-table kernel pads all tables at once
        FK_TIMED("fk_pad_g", s) fk::fk_pad_g_kernel<T><<<(int)std::min<long long>(4096, (tg + 255) / 256), 256, 0, s>>>(g_cat, gP, (int)g->rows_total, R, r0, RP);
        fk::GemmVjpParams p;
        memset(&p, 0, sizeof p);
        p.gP = gP;
        p.G = G;
        p.RP = RP;
        p.nfrag = RP / 8;
        p.nfw = (p.nfrag + 1) / 2;
        p.descs = g->d_descs;
        p.items = g->d_vitems;
        if (g->wsv_all) {
            fk::WsVjpParams w;
            memset(&w, 0, sizeof w);
            w.gP = gP;
            w.G = G;
            w.RP = RP;
            w.ntiles = g->nvitems;
            w.descs = g->d_descs;
            w.items = g->d_vitems;
            if (!wsv_launch<true, TS>(w, s)) return fail(FK_ERR_CUDA, "grouped gemm vjp: cannot reserve %zu bytes of shared memory", fk::WSV_SMEM_BYTES);
        } else if (g->all_vec) FK_TIMED("fk_gemm_vjp", s) fk::fk_gemm_vjp_kernel<2, true><<<g->nvitems, fk::GEMM_THREADS, fk::GEMMV_SMEM_BYTES, s>>>(p);
        else FK_TIMED("fk_gemm_vjp", s) fk::fk_gemm_vjp_kernel<1, true><<<g->nvitems, fk::GEMM_THREADS, fk::GEMMV_SMEM_BYTES, s>>>(p);
        if (g->fold_all) {
            fk::FoldParams q;
            memset(&q, 0, sizeof q);
            q.fT = fT;
            q.G = G;
            q.PA = G + (size_t)g->K_total * RPmax;
            q.PB = q.PA + (size_t)g->cx_total * fk::FOLD_JQ * RPmax;
            q.df = df_cat;
            q.R = R;
            q.r0 = r0;
            q.RP = RP;
            q.nchunk = g->fold_nchunk;
            q.descs = g->d_descs;
            q.items = g->d_foitems;
            q.ai_prefix = g->d_ai_prefix;
            q.T = g->T;
            q.nslots = fk::fold_slots(g->nx_max, RP, MAX_DYN_SMEM);
            if (!ensure_dyn_smem(fk::fk_vjp_fold_kernel<true>, MAX_DYN_SMEM) || q.nslots < 1) return fail(FK_ERR_CUDA, "grouped gemm vjp: cannot reserve shared memory for the fold ring");
            FK_TIMED("fk_vjp_fold", s) fk::fk_vjp_fold_kernel<true><<<g->nfoitems, fk::FOLD_THREADS,
                                           (size_t)q.nslots * g->nx_max * RP * 8 + 2 * fk::FOLD_MAX_SLOTS * 8, s>>>(q);
            FK_TIMED("fk_vjp_fold_final", s) fk::fk_vjp_fold_final_kernel<T, true><<<(unsigned)g->ai_total, fk::GEMM_BN, 0, s>>>(q);
            ++nl;
        } else {
            fk::GatherRParams q;
            memset(&q, 0, sizeof q);
            q.fT = fT;
            q.G = G;
            q.df = df_cat;
            q.R = R;
            q.r0 = r0;
            q.RP = RP;
            q.descs = g->d_descs;
            q.ai_prefix = g->d_ai_prefix;
            q.T = g->T;
            FK_TIMED("fk_vjp_gather_r", s) fk::fk_vjp_gather_r_kernel<T, true><<<dim3((unsigned)g->ai_total, (RP + 127) / 128), 128, 0, s>>>(q);
        }
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "grouped gemm vjp launch failed: %s", cudaGetErrorString(e));
        nl += 4;
    }
    g->last_launches = nl;
    return FK_OK;
}

template <typename T, typename TS = T>
int group_conv_t(fk_group* g, const void* f_cat, void* sigma_cat, int R, cudaStream_t s) {
    int rc = group_scratch(g, group_scratch_need(g, R), s);
    if (rc) return rc;
    if constexpr (std::is_same<T, double>::value) {
        if constexpr (std::is_same<TS, float>::value) {
            if (group_fwd32_wanted(g, R)) return group_conv_gemm<float>(g, (const double*)f_cat, (double*)sigma_cat, R, s);
        }
        if (group_gemm_wanted(g, R)) return group_conv_gemm<double>(g, (const double*)f_cat, (double*)sigma_cat, R, s);
    }
    if constexpr (std::is_same<T, float>::value && std::is_same<TS, float>::value) {
        if (group_tc32_wanted(g, R)) return group_conv_tc32(g, (const float*)f_cat, (float*)sigma_cat, R, s);
    }
    int nl = 0;
    fk::FwdParams p;
    memset(&p, 0, sizeof p);
    p.descs = g->d_descs;
    p.segs = g->d_fsegs;
    p.f = f_cat;
    p.part = g->scratch;
    p.sigma = sigma_cat;
    p.R = R;
    const bool l2_in_kernel = g->d_l2cnt != nullptr && opt(FK_OPT_FUSE_L2) && g->nfsegs <= 8 * std::max(1, sm_count());   // small groups only (fk_api.cu, run_conv_single)
    p.cnt = l2_in_kernel ? g->d_l2cnt : nullptr;
    for (int r0 = 0; r0 < R;) {
        const int rt = pick_rt(R - r0);
        p.r0 = r0;
        cudaError_t e = fwd_dispatch<T, true, TS>(g->all_vec, rt, p, g->nfsegs, s);
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "grouped forward launch failed: %s", cudaGetErrorString(e));
        ++nl;
        r0 += rt;
    }
    if (g->part_total1 > 0 && !l2_in_kernel) {
        fk::ReduceParams q;
        memset(&q, 0, sizeof q);
        q.descs = g->d_descs;
        q.row_prefix = g->d_row_prefix;
        q.T = g->T;
        q.part = g->scratch;
        q.sigma = sigma_cat;
        q.rows = g->rows_total;
        q.R = R;
        const long long outs = g->rows_total * R;
        const int grid = (int)std::min<long long>((outs + 7) / 8, (long long)sm_count() * 8);
        FK_TIMED("fk_reduce_chunks", s) launch_pdl(fk::fk_reduce_chunks_kernel<T, true>, std::max(1, grid), 256, 0, s, q);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "grouped reduce launch failed: %s", cudaGetErrorString(e));
        ++nl;
    }
    g->last_launches = nl;
    return FK_OK;
}

template <typename T, typename TS = T>
int group_vjp_t(fk_group* g, const void* f_cat, const void* g_cat, void* df_cat, int R, cudaStream_t s) {
    int rc = group_scratch(g, group_scratch_need(g, R), s);
    if (rc) return rc;
    if constexpr (std::is_same<TS, double>::value) {
        if (group_gemm_wanted(g, R))
            return group_vjp_gemm<double, double>(g, (const double*)f_cat, (const double*)g_cat, (double*)df_cat, R, s);
    } else {
        if (group_vjp32_wanted(g, R)) return group_vjp_gemm<T, TS>(g, (const T*)f_cat, (const T*)g_cat, (T*)df_cat, R, s);
    }
    int nl = 0;
    fk::ColsumParams p;
    memset(&p, 0, sizeof p);
    p.descs = g->d_descs;
    p.segs = g->d_csegs;
    p.g = g_cat;
    p.G = g->scratch;
    p.R = R;
    for (int r0 = 0; r0 < R;) {
        const int rt = pick_rt(R - r0);
        p.r0 = r0;
        cudaError_t e = colsum_dispatch<T, true, TS>(g->all_vec, rt, p, g->ncsegs, s);
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "grouped colsum launch failed: %s", cudaGetErrorString(e));
        ++nl;
        r0 += rt;
    }
    if (g->foldk_all) {
        if (!ensure_dyn_smem(fk::fk_vjp_foldk_kernel<T, true>, foldk_smem(128)))
            return fail(FK_ERR_CUDA, "grouped vjp: cannot reserve %zu bytes of shared memory", foldk_smem(128));
        fk::FoldKParams q;
        memset(&q, 0, sizeof q);
        q.descs = g->d_descs;
        q.items = g->d_kitems;
        q.ai_prefix = g->d_ai_prefix;
        q.T = g->T;
        q.f = f_cat;
        q.G = g->scratch;
        q.cx_total = g->cx_total;
        q.PA = g->scratch + (size_t)g->G_total1 * R;
        q.PB = q.PA + (size_t)g->cx_total * R;
        q.nchunk = foldk_chunks(g->nkitems);
        q.df = df_cat;
        q.R = R;
        FK_TIMED("fk_vjp_foldk", s) launch_pdl(fk::fk_vjp_foldk_kernel<T, true>, dim3((unsigned)(g->nkitems * q.nchunk), R), fk::FOLDK_THREADS, foldk_smem(g->nx_max), s, q);
        FK_TIMED("fk_vjp_foldk_final", s) launch_pdl(fk::fk_vjp_foldk_final_kernel<T, true>, dim3((unsigned)((g->ai_total + 7) / 8), R), 256, 0, s, q, g->ai_total);
        ++nl;
    } else {
        fk::GatherParams q;
        memset(&q, 0, sizeof q);
        q.descs = g->d_descs;
        q.ai_prefix = g->d_ai_prefix;
        q.T = g->T;
        q.f = f_cat;
        q.G = g->scratch;
        q.df = df_cat;
        q.R = R;
        FK_TIMED("fk_vjp_gather", s) fk::fk_vjp_gather_kernel<T, true><<<dim3((unsigned)g->ai_total, R), fk::GATHER_THREADS, 0, s>>>(q);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(FK_ERR_CUDA, "grouped gather launch failed: %s", cudaGetErrorString(e));
    ++nl;
    g->last_launches = nl;
    return FK_OK;
}

// forward + VJP of the whole group from ONE read of every table (g known before the forward pass, e.g.
// config 4's seeded weights): one fused column launch per <= 4 replicas, the level-2 reduce, the one-pass fold.
template <typename T, typename TS = T>
int group_conv_vjp_fused_t(fk_group* g, const void* f_cat, const void* g_cat, void* sigma_cat, void* df_cat, int R, cudaStream_t s) {
    constexpr int VW = fk::VecWidth<TS>::value;
    int rc = group_scratch(g, group_fused_scratch_need(g, R), s);
    if (rc) return rc;
    double* part = g->scratch;
    double* G = part + (size_t)g->part_total1 * R;
    int nl = 0;
    fk::FusedParams p;
    memset(&p, 0, sizeof p);
    p.fwd.descs = g->d_descs_fused;
    p.fwd.segs = g->d_usegs;
    p.fwd.f = f_cat;
    p.fwd.part = part;
    p.fwd.sigma = sigma_cat;
    p.fwd.R = R;
    p.g = g_cat;
    p.G = G;
    for (int r0 = 0; r0 < R;) {
        const int rt = pick_rt(R - r0);
        p.fwd.r0 = r0;
#define FK_FUSED_G(V, RTv) FK_TIMED("fk_fused_column", s) fk::fk_fused_column_kernel<T, V, RTv, FWD_U, true, TS><<<g->nusegs, fk::FWD_THREADS, 0, s>>>(p)
        if (g->all_vec) {
            if (rt == 1) FK_FUSED_G(VW, 1); else if (rt == 2) FK_FUSED_G(VW, 2); else FK_FUSED_G(VW, 4);
        } else {
            if (rt == 1) FK_FUSED_G(1, 1); else if (rt == 2) FK_FUSED_G(1, 2); else FK_FUSED_G(1, 4);
        }
#undef FK_FUSED_G
        ++nl;
        r0 += rt;
    }
    if (g->part_total1 > 0) {
        fk::ReduceParams q;
        memset(&q, 0, sizeof q);
        q.descs = g->d_descs_fused;
        q.row_prefix = g->d_row_prefix;
        q.T = g->T;
        q.part = part;
        q.sigma = sigma_cat;
        q.rows = g->rows_total;
        q.R = R;
        const long long outs = g->rows_total * R;
        const int grid = (int)std::min<long long>((outs + 7) / 8, (long long)sm_count() * 8);
        FK_TIMED("fk_reduce_chunks", s) launch_pdl(fk::fk_reduce_chunks_kernel<T, true>, std::max(1, grid), 256, 0, s, q);
        ++nl;
    }
    if (!ensure_dyn_smem(fk::fk_vjp_foldk_kernel<T, true>, foldk_smem(128)))
        return fail(FK_ERR_CUDA, "grouped conv_vjp: cannot reserve %zu bytes of shared memory", foldk_smem(128));
    fk::FoldKParams q;
    memset(&q, 0, sizeof q);
    q.descs = g->d_descs_fused;
    q.items = g->d_kitems;
    q.ai_prefix = g->d_ai_prefix;
    q.T = g->T;
    q.f = f_cat;
    q.G = G;
    q.cx_total = g->cx_total;
    q.PA = G + (size_t)g->G_total1_fused * R;
    q.PB = q.PA + (size_t)g->cx_total * R;
    q.nchunk = foldk_chunks(g->nkitems);
    q.df = df_cat;
    q.R = R;
    FK_TIMED("fk_vjp_foldk", s) launch_pdl(fk::fk_vjp_foldk_kernel<T, true>, dim3((unsigned)(g->nkitems * q.nchunk), R), fk::FOLDK_THREADS, foldk_smem(g->nx_max), s, q);
    FK_TIMED("fk_vjp_foldk_final", s) launch_pdl(fk::fk_vjp_foldk_final_kernel<T, true>, dim3((unsigned)((g->ai_total + 7) / 8), R), 256, 0, s, q, g->ai_total);
    nl += 2;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(FK_ERR_CUDA, "grouped fused forward + VJP launch failed: %s", cudaGetErrorString(e));
    g->last_launches = nl;
    return FK_OK;
}

template <typename T, typename TS = T>
int group_conv_vjp_t(fk_group* g, const void* f_cat, const void* g_cat, void* sigma_cat, void* df_cat, int R, cudaStream_t s) {
    if (group_fused_wanted(g, R)) return group_conv_vjp_fused_t<T, TS>(g, f_cat, g_cat, sigma_cat, df_cat, R, s);
    int rc = group_conv_t<T, TS>(g, f_cat, sigma_cat, R, s);   // two passes: R >= 5, DIS tables, very large x-grids
    if (rc) return rc;
    const int nl = g->last_launches;
    rc = group_vjp_t<T, TS>(g, f_cat, g_cat, df_cat, R, s);
    g->last_launches += nl;
    return rc;
}

}  // namespace

extern "C" {

int fk_group_create(fk_group** out, fk_table* const* tables, int T, int R_hint) {
    g_err.clear();
    if (!out) return fail(FK_ERR_INVALID_ARG, "fk_group_create: null out");
    *out = nullptr;
    if (!tables || T <= 0) return fail(FK_ERR_INVALID_ARG, "fk_group_create: no tables");
    for (int t = 0; t < T; ++t)
        if (!tables[t]) return fail(FK_ERR_INVALID_ARG, "fk_group_create: table %d is null", t);
    fk_group* g = new (std::nothrow) fk_group();
    if (!g) return fail(FK_ERR_ALLOC, "fk_group_create: host allocation failed");
    g->T = T;
    g->dtype = tables[0]->dtype;
    if (g->sync.init() != FK_OK) { delete g; return fail(FK_ERR_CUDA, "fk_group_create: no CUDA device"); }
    std::vector<int> row_prefix(T + 1, 0), ai_prefix(T + 1, 0);
    for (int t = 0; t < T; ++t) {
        fk_table* tb = tables[t];
        if (tb->dtype != g->dtype) { g->sync.destroy(); delete g; return fail(FK_ERR_INVALID_ARG, "fk_group_create: mixed dtypes"); }
        if (tb->sync.device != g->sync.device) {
            g->sync.destroy(); delete g;
            return fail(FK_ERR_INVALID_ARG, "fk_group_create: table %d lives on device %d, the current device is %d", t, tb->sync.device, g->sync.device);
        }
        if (tb->desc.sp_blk) {
            g->sync.destroy(); delete g;
            return fail(FK_ERR_UNSUPPORTED, "fk_group_create: table %d uses sparse storage, which the grouped launch does not take", t);
        }
        g->all_vec = g->all_vec && tb->desc.vec_ok;
    }
    // R >> 1 contraction: every item (128-datapoint tile x K range) costs about the same DMMA time
    g->gemm_ok = g->dtype == FK_F64;
    long long tile_k = 0;
    for (int t = 0; t < T; ++t) {
        g->gemm_ok = g->gemm_ok && tables[t]->kdec != nullptr;
        tile_k += (long long)((tables[t]->desc.N + fk::GEMM_BM - 1) / fk::GEMM_BM) * tables[t]->desc.K;
    }
    const long long want_items = (long long)std::max(1, sm_count()) * GROUP_GEMM_WAVES;
    long long kper_target = (tile_k + want_items - 1) / want_items;
    kper_target = std::max<long long>(fk::GEMM_KT * 8, (kper_target + fk::GEMM_KT - 1) / fk::GEMM_KT * fk::GEMM_KT);
    std::vector<fk::ColSeg> fsegs, csegs, gitems, vitems, foitems, witems, kitems, usegs;
    std::vector<fk::TableDesc> descs_fused;
    long long group_kblocks = 0;
    for (int t = 0; t < T; ++t) group_kblocks += tables[t]->desc.nchunks;
    {
        long long channels = 0;
        for (int t = 0; t < T; ++t) channels += tables[t]->desc.C;
        g->fold_nchunk = fold_chunks(channels);
    }
    for (int t = 0; t < T; ++t) {
        fk_table* tb = tables[t];
        fk::TableDesc d = tb->desc;
        {
            const int ksplit0 = (int)std::max<long long>(1, (d.K + kper_target - 1) / kper_target);
            d.gkper = ((d.K + ksplit0 - 1) / ksplit0 + fk::GEMM_KT - 1) / fk::GEMM_KT * fk::GEMM_KT;
            d.gksplit = (d.K + d.gkper - 1) / d.gkper;
            // a partial last datapoint tile is cut into k sub-splits that take whole groups of K ranges
            // (65..96 remaining datapoints take a 64-row and a 32-row tile instead of a 128-row one)
            const int nfull = d.N / fk::GEMM_BM, rem = d.N % fk::GEMM_BM;
            const bool two = rem > 64 && rem <= 96;
            const int ksub_rem = rem ? (two ? 4 : fk::ws_ksub_for_rows(rem)) : 1;
            d.gksplit = (d.gksplit + ksub_rem - 1) / ksub_rem * ksub_rem;
            for (int ks = 0; ks < d.gksplit; ++ks)
                for (int mt = 0; mt < nfull; ++mt) witems.push_back(fk::ColSeg{t, mt * fk::GEMM_BM, ks, 1});
            if (two) {
                for (int ks = 0; ks < d.gksplit / 2; ++ks) witems.push_back(fk::ColSeg{t, nfull * fk::GEMM_BM, ks, 2});
                for (int ks = 0; ks < d.gksplit / 4; ++ks) witems.push_back(fk::ColSeg{t, nfull * fk::GEMM_BM + 64, ks, 4});
            } else if (rem) {
                for (int ks = 0; ks < d.gksplit / ksub_rem; ++ks) witems.push_back(fk::ColSeg{t, nfull * fk::GEMM_BM, ks, ksub_rem});
            }
            g->ws_all = g->ws_all && d.kind == fk::KIND_HADRONIC && d.layout == fk::LAYOUT_PACKED && d.vec_ok;
            g->jp_all = g->jp_all && d.jp == d.nx;
            g->nx_max = std::max(g->nx_max, d.nx);
            d.gp_off = g->gp_rows;
            d.k_off = g->K_total;
            g->gp_rows += (long long)d.gksplit * d.N;
            g->K_total += d.K;
            const int mtiles = (d.N + fk::GEMM_BM - 1) / fk::GEMM_BM;
            for (int ks = 0; ks < d.gksplit; ++ks)
                for (int mt = 0; mt < mtiles; ++mt) gitems.push_back(fk::ColSeg{t, mt, ks, 0});
            for (int kt = 0; kt < (d.K + fk::GEMMV_BK - 1) / fk::GEMMV_BK; ++kt) vitems.push_back(fk::ColSeg{t, kt, 0, 0});
            d.cx_off = g->cx_total;
            g->cx_total += (long long)d.C * d.nx;
            g->fold_all = g->fold_all && fold_ok(d);
            g->wsv_all = g->wsv_all && wsv_ok(d);
            g->foldk_all = g->foldk_all && foldk_ok(d);
            for (int c = 0; c < d.C; ++c) kitems.push_back(fk::ColSeg{t, c, 0, 0});
            for (int c = 0; c < d.C; ++c)
                for (int ch = 0; ch < g->fold_nchunk; ++ch) foitems.push_back(fk::ColSeg{t, c, ch, 0});
        }
        if (!g->all_vec && d.vec_ok) {  // one kernel instantiation per launch: the whole group takes the 64-bit path
            d.vec_ok = 0;
            Plan pl;
            make_plan(d, g->dtype, pl);
        }
        {   // VJP stage 1: the GROUP has to fill the GPU, not every table on its own -- fewer datapoint ranges per
            // k-block mean fewer column-sum slices G[nsplit][R][K] to write and to gather (a table planned alone asks
            // for ~24 CTAs per SM and gets up to N/16 slices)
            const long long want = (long long)COLSUM_CTAS_PER_SM * std::max(1, sm_count());
            int ns = (int)std::min<long long>(std::max<long long>(1, (want + group_kblocks - 1) / std::max<long long>(1, group_kblocks)),
                                              std::max(1, d.N / 16));
            ns = std::max(ns, (d.N + fk::COLSUM_MAX_ROWS - 1) / fk::COLSUM_MAX_ROWS);
            d.nsplit = std::max(1, std::min(ns, d.N));
        }
        d.cnt_off = g->cnt_total;
        g->cnt_total += d.fsplit;
        d.f_off = g->f_total1;
        d.out_off = g->rows_total;
        d.part_off = g->part_total1;
        d.g_off = g->G_total1;
        g->f_total1 += (long long)d.nfl * d.nx;
        g->rows_total += d.N;
        g->ai_total += (long long)d.nfl * d.nx;
        g->part_total1 += (long long)part_elems_per_replica(d);
        g->G_total1 += (long long)G_elems_per_replica(d);
        g->elems_total += (long long)d.N * d.K;
        row_prefix[t + 1] = (int)g->rows_total;
        ai_prefix[t + 1] = (int)g->ai_total;
        for (int sp = 0; sp < d.fsplit; ++sp)
            for (int kb = 0; kb < d.nchunks; ++kb) fsegs.push_back(fk::ColSeg{t, kb, sp, 0});
        for (int sp = 0; sp < d.nsplit; ++sp)
            for (int kb = 0; kb < d.nchunks; ++kb) csegs.push_back(fk::ColSeg{t, kb, sp, 0});
        g->tables.push_back(tb);
        g->descs.push_back(d);
        {   // one-read forward + VJP: up to 64 datapoints per CTA; its ranges are the slices of the column sums
            fk::TableDesc du = d;
            du.fsplit = std::max(1, std::min(d.fsplit, (d.N + 63) / 64));
            du.nsplit = du.fsplit;
            du.g_off = g->G_total1_fused;
            g->G_total1_fused += (long long)du.fsplit * du.K;
            g->fused_all = g->fused_all && foldk_ok(du) && (du.N + du.fsplit - 1) / du.fsplit <= 64;
            for (int sp = 0; sp < du.fsplit; ++sp)
                for (int kb = 0; kb < du.nchunks; ++kb) usegs.push_back(fk::ColSeg{t, kb, sp, 0});
            descs_fused.push_back(du);
        }
    }
    std::vector<fk::ColSeg> tcitems;
    if (g->dtype == FK_F32) {   // tcgen05 items of about equal cost: 4 waves of (128-datapoint tile) x (range of (c, i) rows)
        g->tc_all = true;
        long long work = 0;
        for (int t = 0; t < T; ++t) {
            const fk::TableDesc& d = g->descs[t];
            g->tc_all = g->tc_all && d.tmap && d.kind == fk::KIND_HADRONIC && d.layout == fk::LAYOUT_PACKED && d.nx <= fk::TC_MAX_NX && d.jp % 4 == 0;
            work += (long long)fk::tc32_ntiles(d.N) * d.C * d.nx;
        }
        if (g->tc_all) {
            const long long tper_target = std::max<long long>(16, (work + 4LL * std::max(1, sm_count()) - 1) / (4LL * std::max(1, sm_count())));
            for (int t = 0; t < T; ++t) {
                fk::TableDesc& d = g->descs[t];
                const int Trows = d.C * d.nx;
                int ksplit = (int)std::max<long long>(1, (Trows + tper_target - 1) / tper_target);
                ksplit = std::max(ksplit, (Trows + fk::TC_MAX_TILES - 1) / fk::TC_MAX_TILES);
                d.tc_kper = (Trows + ksplit - 1) / ksplit;
                d.tc_ksplit = (Trows + d.tc_kper - 1) / d.tc_kper;
                d.tc_gp_off = g->tc_gp_rows;
                g->tc_gp_rows += (long long)d.tc_ksplit * d.N;
                for (int ks = 0; ks < d.tc_ksplit; ++ks)
                    for (int n0 = 0; n0 < d.N; n0 += fk::TC_BN) tcitems.push_back(fk::ColSeg{t, n0, ks, 0});
            }
        }
    }
    g->ntcitems = (int)tcitems.size();
    if (g->rows_total >= (1LL << 31) || g->ai_total >= (1LL << 31)) {
        g->sync.destroy();
        delete g;
        return fail(FK_ERR_UNSUPPORTED, "fk_group_create: more than 2^31 datapoints or PDF slots");
    }
    g->nfsegs = (int)fsegs.size();
    g->ncsegs = (int)csegs.size();
    g->ngitems = (int)gitems.size();
    g->nvitems = (int)vitems.size();
    g->nfoitems = (int)foitems.size();
    g->nwitems = (int)witems.size();
    g->nkitems = (int)kitems.size();
    g->nusegs = (int)usegs.size();
    auto bail = [&](int code) { fk_group_destroy(g); return code; };
    cudaError_t e = cudaMalloc((void**)&g->d_descs, T * sizeof(fk::TableDesc));
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_row_prefix, (T + 1) * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_ai_prefix, (T + 1) * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_csegs, csegs.size() * sizeof(fk::ColSeg));
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_fsegs, fsegs.size() * sizeof(fk::ColSeg));
    if (e == cudaSuccess) e = cudaMemcpy(g->d_fsegs, fsegs.data(), fsegs.size() * sizeof(fk::ColSeg), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_gitems, gitems.size() * sizeof(fk::ColSeg));
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_vitems, vitems.size() * sizeof(fk::ColSeg));
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_foitems, foitems.size() * sizeof(fk::ColSeg));
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_kitems, kitems.size() * sizeof(fk::ColSeg));
    if (e == cudaSuccess) e = cudaMemcpy(g->d_kitems, kitems.data(), kitems.size() * sizeof(fk::ColSeg), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_witems, std::max<size_t>(1, witems.size()) * sizeof(fk::ColSeg));
    if (e == cudaSuccess) e = cudaMemcpy(g->d_witems, witems.data(), witems.size() * sizeof(fk::ColSeg), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(g->d_foitems, foitems.data(), foitems.size() * sizeof(fk::ColSeg), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(g->d_gitems, gitems.data(), gitems.size() * sizeof(fk::ColSeg), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(g->d_vitems, vitems.data(), vitems.size() * sizeof(fk::ColSeg), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(g->d_descs, g->descs.data(), T * sizeof(fk::TableDesc), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(g->d_row_prefix, row_prefix.data(), (T + 1) * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(g->d_ai_prefix, ai_prefix.data(), (T + 1) * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(g->d_csegs, csegs.data(), csegs.size() * sizeof(fk::ColSeg), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_l2cnt, (size_t)std::max<long long>(1, g->cnt_total) * sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(g->d_l2cnt, 0, (size_t)std::max<long long>(1, g->cnt_total) * sizeof(int));
    if (e == cudaSuccess && !tcitems.empty()) e = cudaMalloc((void**)&g->d_tcitems, tcitems.size() * sizeof(fk::ColSeg));
    if (e == cudaSuccess && !tcitems.empty()) e = cudaMemcpy(g->d_tcitems, tcitems.data(), tcitems.size() * sizeof(fk::ColSeg), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_descs_fused, T * sizeof(fk::TableDesc));
    if (e == cudaSuccess) e = cudaMemcpy(g->d_descs_fused, descs_fused.data(), T * sizeof(fk::TableDesc), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_usegs, usegs.size() * sizeof(fk::ColSeg));
    if (e == cudaSuccess) e = cudaMemcpy(g->d_usegs, usegs.data(), usegs.size() * sizeof(fk::ColSeg), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { bail(0); return fail(FK_ERR_CUDA, "fk_group_create: %s", cudaGetErrorString(e)); }
    int rc = group_scratch(g, std::max(group_scratch_need(g, 1), group_scratch_need(g, std::max(1, R_hint))));
    if (rc) return bail(rc);
    *out = g;
    return FK_OK;
}

int fk_group_destroy(fk_group* g) {
    if (!g) return FK_OK;
    if (g->d_descs) cudaFree(g->d_descs);
    if (g->d_row_prefix) cudaFree(g->d_row_prefix);
    if (g->d_ai_prefix) cudaFree(g->d_ai_prefix);
    if (g->d_csegs) cudaFree(g->d_csegs);
    if (g->d_fsegs) cudaFree(g->d_fsegs);
    if (g->d_gitems) cudaFree(g->d_gitems);
    if (g->d_vitems) cudaFree(g->d_vitems);
    if (g->d_foitems) cudaFree(g->d_foitems);
    if (g->d_kitems) cudaFree(g->d_kitems);
    if (g->d_witems) cudaFree(g->d_witems);
    if (g->d_tcitems) cudaFree(g->d_tcitems);
    if (g->d_l2cnt) cudaFree(g->d_l2cnt);
    if (g->d_descs_fused) cudaFree(g->d_descs_fused);
    if (g->d_usegs) cudaFree(g->d_usegs);
    if (g->scratch) cudaFree(g->scratch);
    g->sync.destroy();
    delete g;
    return FK_OK;
}

int fk_group_offsets(const fk_group* g, int R, int64_t* f_offsets, int64_t* sigma_offsets) {
    if (!g || R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_group_offsets: bad argument");
    for (int t = 0; t < g->T; ++t) {
        if (f_offsets) f_offsets[t] = g->descs[t].f_off * R;
        if (sigma_offsets) sigma_offsets[t] = g->descs[t].out_off * R;
    }
    if (f_offsets) f_offsets[g->T] = g->f_total1 * R;
    if (sigma_offsets) sigma_offsets[g->T] = g->rows_total * R;
    return FK_OK;
}

int fk_conv_grouped(fk_group* g, const void* f_cat, void* sigma_cat, int R, void* stream) {
    g_err.clear();
    if (!g || !f_cat || !sigma_cat) return fail(FK_ERR_INVALID_ARG, "fk_conv_grouped: null pointer");
    if (R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_conv_grouped: R=%d", R);
    CallGuard cg(g->sync, (cudaStream_t)stream);
    if (int rc = cg.begin("fk_conv_grouped")) return rc;
    if (g->dtype == FK_F32S64) return group_conv_t<double, float>(g, f_cat, sigma_cat, R, (cudaStream_t)stream);
    return g->dtype == FK_F64 ? group_conv_t<double>(g, f_cat, sigma_cat, R, (cudaStream_t)stream)
                              : group_conv_t<float>(g, f_cat, sigma_cat, R, (cudaStream_t)stream);
}

int fk_conv_grouped_vjp(fk_group* g, const void* f_cat, const void* g_cat, void* df_cat, int R, void* stream) {
    g_err.clear();
    if (!g || !f_cat || !g_cat || !df_cat) return fail(FK_ERR_INVALID_ARG, "fk_conv_grouped_vjp: null pointer");
    if (R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_conv_grouped_vjp: R=%d", R);
    CallGuard cg(g->sync, (cudaStream_t)stream);
    if (int rc = cg.begin("fk_conv_grouped_vjp")) return rc;
    if (g->dtype == FK_F32S64) return group_vjp_t<double, float>(g, f_cat, g_cat, df_cat, R, (cudaStream_t)stream);
    return g->dtype == FK_F64 ? group_vjp_t<double>(g, f_cat, g_cat, df_cat, R, (cudaStream_t)stream)
                              : group_vjp_t<float>(g, f_cat, g_cat, df_cat, R, (cudaStream_t)stream);
}

int fk_conv_grouped_conv_vjp(fk_group* g, const void* f_cat, const void* g_cat, void* sigma_cat, void* df_cat, int R, void* stream) {
    g_err.clear();
    if (!g || !f_cat || !g_cat || !sigma_cat || !df_cat) return fail(FK_ERR_INVALID_ARG, "fk_conv_grouped_conv_vjp: null pointer");
    if (R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_conv_grouped_conv_vjp: R=%d", R);
    cudaStream_t s = (cudaStream_t)stream;
    CallGuard cg(g->sync, s);
    if (int rc = cg.begin("fk_conv_grouped_conv_vjp")) return rc;
    if (g->dtype == FK_F32S64) return group_conv_vjp_t<double, float>(g, f_cat, g_cat, sigma_cat, df_cat, R, s);
    return g->dtype == FK_F64 ? group_conv_vjp_t<double>(g, f_cat, g_cat, sigma_cat, df_cat, R, s)
                              : group_conv_vjp_t<float>(g, f_cat, g_cat, sigma_cat, df_cat, R, s);
}

int fk_group_last_launches(const fk_group* g) { return g ? g->last_launches : 0; }

}  // extern "C"
