// qw_step_tiled2d_host.cuh — host-side launcher of step_tiled2d_kernel for ONE dtype; included by
// qw_step_tiled2d_f32.cu / _f64.cu (one translation unit per dtype keeps the build parallel).
#pragma once

#include "qw_step_tiled2d.cuh"

namespace qw {

typedef CUresult (*T2dEncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static T2dEncodeFn t2d_encode_fn() {
    static T2dEncodeFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<T2dEncodeFn>(p);
    }
    return fn;
}

// One tensor map per state buffer: (n in 8-byte words, padded rows, plane * batch + walk), box = one tile of one plane.
template <typename R>
static int t2d_build_tmaps(qw_sim *s) {
    if (s->tmap_t_ready) return QW_OK;
    typedef T2dCfg<R> G;
    T2dEncodeFn enc = t2d_encode_fn();
    if (!enc) return fail(QW_ECUDA, "cuTensorMapEncodeTiled is not available from this driver");
    const Geom &g = s->g;
    const cuuint64_t words = s->esize / 8;
    const cuuint64_t dims[3] = {(cuuint64_t)g.pitch * words, (cuuint64_t)(g.em + 2 * g.ghost), (cuuint64_t)(4 * g.batch)};
    const cuuint64_t strides[2] = {(cuuint64_t)g.pitch * s->esize, (cuuint64_t)g.walk_stride * s->esize};
    const cuuint32_t box[3] = {(cuuint32_t)(32 * G::RN * words), (cuuint32_t)(G::W * G::RM), 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    for (int i = 0; i < 2; ++i) {
        CUresult r = enc(reinterpret_cast<CUtensorMap *>(s->tmap_t[i]), CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, s->buf[i], dims, strides,
                         box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(QW_ECUDA, "cuTensorMapEncodeTiled failed with code %d", (int)r);
    }
    s->tmap_t_ready = true;
    return QW_OK;
}

template <typename R, int KIND, int K>
static int t2d_launch_k(qw_sim *s, int in_buf, int out_buf, const Box &box) {
    typedef typename Cx<R>::T V;
    typedef T2dCfg<R> G;
    constexpr int HM = G::W * G::RM, HN = 32 * G::RN, TM = HM - 2 * K, TN = HN - 2 * K;
    const Geom &g = s->g;
    Tiled2dArgs<R> a;
    a.out = static_cast<V *>(state_ptr(s, out_buf));
    a.em = g.em; a.en = g.en; a.pitch = g.pitch; a.walk_stride = g.walk_stride; a.plane_stride = g.plane_stride;
    a.batch = (int)g.batch; a.ghost = g.ghost;
    // tiles of the global grid whose valid interior meets the box of sites that can be non-zero afterwards
    a.tile_m0 = (int)(box.m_lo / TM); a.tile_n0 = (int)(box.n_lo / TN);
    a.tiles_m = (int)(box.m_hi / TM) - a.tile_m0 + 1; a.tiles_n = (int)(box.n_hi / TN) - a.tile_n0 + 1;
    a.total_tiles = (long long)a.tiles_m * a.tiles_n * g.batch;
    for (int i = 0; i < 32; ++i) a.coin[i] = (R)s->h_coin[i];
    // deferred scale (named coins only; their scale is a power of two, so every product below is exact)
    const double scale = KIND == COIN_GROVER4 ? s->h_coin[2] : s->h_coin[0];
    double pw = 1.0;
    for (int i = 0; i < K - 1; ++i) pw *= scale;
    for (int i = 0; i < 32; ++i) a.coin_last[i] = (R)(s->h_coin[i] * pw);
    a.ratio = KIND == COIN_GROVER4 ? (R)((s->h_coin[0] - s->h_coin[2]) / s->h_coin[2]) : (R)0;
    // diamond of the light cone after this launch; on a torus only while the square box has not wrapped
    a.dia_r = -1; a.dia_m = s->centre[0]; a.dia_n = s->centre[1];
    const bool diag = g.lattice == QW_DIAGONAL;      // both coordinates move: the cone is the square, no diamond
    if (!diag && s->window_enabled && s->window_valid) {
        const long long r = s->radius + K;
        const bool wraps = g.boundary == QW_PERIODIC &&
                           (a.dia_m - r < 0 || a.dia_m + r >= g.em || a.dia_n - r < 0 || a.dia_n + r >= g.en);
        if (!wraps) a.dia_r = r;
    }
    const size_t smem = diag ? tiled2d_smem_bytes<R, true>() : tiled2d_smem_bytes<R, false>();
    const long long cap = (long long)s->sm_count;              // persistent: one CTA per SM
    const unsigned grid = (unsigned)(a.total_tiles < cap ? a.total_tiles : cap);
    const CUtensorMap &tm = *reinterpret_cast<const CUtensorMap *>(s->tmap_t[in_buf]);
    auto go = [&](auto kernel) -> int {
        QW_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kernel<<<grid, G::W * 32, smem, s->stream>>>(tm, a);
        return QW_OK;
    };
    // diagonal lattice: no wall code in the kernel; the dispatcher only comes here when no amplitude can touch a wall
    int rc = diag ? go(step_tiled2d_kernel<R, KIND, false, K, true>)
                  : (g.boundary == QW_OPEN ? go(step_tiled2d_kernel<R, KIND, true, K>) : go(step_tiled2d_kernel<R, KIND, false, K>));
    if (rc) return rc;
    QW_LAUNCH_CHECK(s, "step_tiled2d_kernel");
    {   // site-steps actually computed: the valid interiors of the tiles the kernel's diamond test leaves active
        double sites = 0.0;
        for (int tm = 0; tm < a.tiles_m; ++tm)
            for (int tn = 0; tn < a.tiles_n; ++tn) {
                const long long lo_m = (long long)(a.tile_m0 + tm) * TM, lo_n = (long long)(a.tile_n0 + tn) * TN;
                if (a.dia_r >= 0) {
                    const long long dm = a.dia_m < lo_m ? lo_m - a.dia_m : (a.dia_m > lo_m + TM - 1 ? a.dia_m - (lo_m + TM - 1) : 0);
                    const long long dn = a.dia_n < lo_n ? lo_n - a.dia_n : (a.dia_n > lo_n + TN - 1 ? a.dia_n - (lo_n + TN - 1) : 0);
                    if (dm + dn > a.dia_r) continue;
                }
                const long long hm = lo_m + TM <= g.em ? TM : g.em - lo_m, hn = lo_n + TN <= g.en ? TN : g.en - lo_n;
                if (hm > 0 && hn > 0) sites += (double)hm * (double)hn;
            }
        s->touched += sites * (double)g.batch * K;
    }
    return QW_OK;
}

template <typename R, int KIND>
static int t2d_launch_kind(qw_sim *s, int in_buf, int out_buf, int k, const Box &box) {
    switch (k) {
        case 2: return t2d_launch_k<R, KIND, 2>(s, in_buf, out_buf, box);
        case 4: return t2d_launch_k<R, KIND, 4>(s, in_buf, out_buf, box);
        case 6: return t2d_launch_k<R, KIND, 6>(s, in_buf, out_buf, box);
        case 8: return t2d_launch_k<R, KIND, 8>(s, in_buf, out_buf, box);
        default: return fail(QW_EINVAL, "tiled 2D step depth %d is not one of 2, 4, 6, 8", k);
    }
}

template <typename R>
static int t2d_launch(qw_sim *s, int in_buf, int out_buf, int k, const Box &box) {
    int rc = t2d_build_tmaps<R>(s);
    if (rc) return rc;
    switch (s->coin_kind) {
        case COIN_GROVER4: return t2d_launch_kind<R, COIN_GROVER4>(s, in_buf, out_buf, k, box);
        case COIN_HXH4:    return t2d_launch_kind<R, COIN_HXH4>(s, in_buf, out_buf, k, box);
        case COIN_DFT4:    return t2d_launch_kind<R, COIN_DFT4>(s, in_buf, out_buf, k, box);
        default:           return t2d_launch_kind<R, COIN_GENERAL>(s, in_buf, out_buf, k, box);
    }
}

}  // namespace qw
