// qw_step_stream2d_host.cuh — host-side launcher of step_stream2d_kernel for ONE dtype; included by
// qw_step_stream2d_f32.cu / _f64.cu (one translation unit per dtype keeps the build parallel).
#pragma once

#include "qw_step_stream2d.cuh"

namespace qw {

// Work units of one launch: (walk, segment of rows, strip of columns), strips fastest, handed to the warps of the
// persistent grid round-robin — so the warps that run at the same time work on neighbouring strips of the same
// rows and the column halos they share are read from HBM once (the second reader hits L2).
struct S2dPlan {
    int strip0, strips, segs;
    long long seg_len;
    double cost;
};

// does the unit with output rows [a0, b0) x columns [n_lo, n_hi] meet the diamond?
static inline bool s2d_unit_active(long long a0, long long b0, long long n_lo, long long n_hi, long long dm0, long long dn0, long long dr) {
    if (dr < 0) return true;
    const long long dm = dm0 < a0 ? a0 - dm0 : (dm0 > b0 - 1 ? dm0 - (b0 - 1) : 0);
    const long long dn = dn0 < n_lo ? n_lo - dn0 : (dn0 > n_hi ? dn0 - n_hi : 0);
    return dm + dn <= dr;
}

// number of strips of the launched range [strip0, strip0 + strips) that meet the diamond in the segment of rows [a0, b0): they
// form one interval (the kernel enumerates it with the same formula)
static inline long long s2d_row_count(long long a0, long long b0, int strip0, int strips, int VN, long long dm0, long long dn0, long long dr) {
    if (a0 >= b0) return 0;
    const long long dm = dm0 < a0 ? a0 - dm0 : (dm0 > b0 - 1 ? dm0 - (b0 - 1) : 0);
    const long long rem = dr - dm;
    if (rem < 0) return 0;
    long long lo = (dn0 - rem) / VN, hi = (dn0 + rem) / VN;
    if (lo < strip0) lo = strip0;
    if (hi > strip0 + strips - 1) hi = strip0 + strips - 1;
    return hi >= lo ? hi - lo + 1 : 0;
}

// Segments per strip: every segment costs seg_len + 2K row cascades (the pipeline fills and drains), the launch takes
// ceil(active units / warps) rounds of them.  Candidates: the segment counts that fill 1 .. 8 rounds of the grid.
static S2dPlan s2d_plan(const Box &box, long long batch, int VN, int K, long long warps, long long dm0, long long dn0, long long dr) {
    S2dPlan best;
    best.strip0 = (int)(box.n_lo / VN);
    best.strips = (int)(box.n_hi / VN) - best.strip0 + 1;
    best.segs = 1; best.seg_len = box.m_hi - box.m_lo + 1; best.cost = -1.0;
    const long long rows = box.m_hi - box.m_lo + 1;
    const long long per_seg = batch * best.strips;
    for (int round = 1; round <= 8; ++round) {
        long long segs = round * warps / per_seg;
        if (segs < 1) segs = 1;
        const long long min_len = 2LL * K;                      // never more fill/drain rows than payload rows
        const bool shortest = segs >= rows / min_len;
        if (shortest) segs = rows / min_len > 0 ? rows / min_len : 1;
        const long long len = (rows + segs - 1) / segs;
        segs = (rows + len - 1) / len;
        long long active = 0;
        if (dr < 0) active = segs * per_seg;
        else
            for (long long sg = 0; sg < segs; ++sg) {
                const long long a0 = box.m_lo + sg * len, b0 = a0 + len <= box.m_hi + 1 ? a0 + len : box.m_hi + 1;
                for (int st = 0; st < best.strips; ++st) {
                    const long long n_lo = (long long)(best.strip0 + st) * VN;
                    if (s2d_unit_active(a0, b0, n_lo, n_lo + VN - 1, dm0, dn0, dr)) active += batch;
                }
            }
        const double cost = (double)((active + warps - 1) / warps) * (double)(len + 2 * K + 2);
        if (best.cost < 0 || cost < best.cost) { best.segs = (int)segs; best.seg_len = len; best.cost = cost; }
        if (shortest) break;                                      // the segments cannot get any shorter
    }
    // With a diamond the active units are dealt round-robin (the kernel enumerates them), so the launch takes
    // ceil(active / warps) rounds: every segment count is a candidate (the active count of a segment row is closed-form).
    if (dr >= 0) {
        const long long max_segs = rows / (2LL * K) > 0 ? rows / (2LL * K) : 1;
        long long prev_len = -1;
        for (long long sg_n = 1; sg_n <= max_segs; ++sg_n) {
            const long long len = (rows + sg_n - 1) / sg_n;
            if (len == prev_len) continue;
            prev_len = len;
            const long long segs = (rows + len - 1) / len;
            long long active = 0;
            for (long long sg = 0; sg < segs; ++sg) {
                const long long a0 = box.m_lo + sg * len, b0 = a0 + len <= box.m_hi + 1 ? a0 + len : box.m_hi + 1;
                active += s2d_row_count(a0, b0, best.strip0, best.strips, VN, dm0, dn0, dr);
            }
            active *= batch;
            const double cost = (double)((active + warps - 1) / warps) * (double)(len + 2 * K + 2);
            if (cost < best.cost) { best.segs = (int)segs; best.seg_len = len; best.cost = cost; }
        }
    }
    return best;
}

template <typename R, int KIND, int K, bool RBL>
static int s2d_launch_k(qw_sim *s, int in_buf, int out_buf, const Box &box) {
    typedef typename Cx<R>::T V;
    constexpr int RN = S2dShape<R, K, RBL>::RN, HN = 32 * RN, VN = HN - 2 * K, WPC = S2dShape<R, K, RBL>::WPC;
    const Geom &g = s->g;
    Stream2dArgs<R> a;
    a.in = static_cast<const V *>(state_ptr(s, in_buf));
    a.out = static_cast<V *>(state_ptr(s, out_buf));
    a.em = g.em; a.en = g.en; a.pitch = g.pitch; a.walk_stride = g.walk_stride; a.plane_stride = g.plane_stride;
    a.max_col = (g.pitch - g.ghost - RN) / RN * RN;
    a.wrap = stream2d_wraps(s) ? 1 : 0;
    a.batch = (int)g.batch;
    for (int i = 0; i < 32; ++i) a.coin[i] = (R)s->h_coin[i];
    // deferred scale (named coins only; their scale is a power of two, so every product below is exact)
    const double scale = KIND == COIN_GROVER4 ? s->h_coin[2] : s->h_coin[0];
    double pw = 1.0;
    for (int i = 0; i < K - 1; ++i) pw *= scale;
    for (int i = 0; i < 32; ++i) a.coin_last[i] = (R)(s->h_coin[i] * pw);
    a.ratio = KIND == COIN_GROVER4 ? (R)((s->h_coin[0] - s->h_coin[2]) / s->h_coin[2]) : (R)0;
    a.rbl_key0 = (unsigned)(s->rbl_seed & 0xffffffffu); a.rbl_key1 = (unsigned)(s->rbl_seed >> 32);
    a.rbl_thr = s->rbl_thr;
    a.t = (unsigned)((unsigned long long)s->t & 0xffffffffu);     // level l of the pipeline = step t + l
    // diamond of the light cone after this launch; on a torus only while the square box has not wrapped
    a.dia_r = -1; a.dia_m = s->centre[0]; a.dia_n = s->centre[1];
    if (s->window_enabled && s->window_valid) {
        const long long r = s->radius + K;
        const bool wraps = g.boundary == QW_PERIODIC &&
                           (a.dia_m - r < 0 || a.dia_m + r >= g.em || a.dia_n - r < 0 || a.dia_n + r >= g.en);
        if (!wraps) a.dia_r = r;
    }
    int ctas = s->sm_count;
    if (s->max_ctas > 0 && s->max_ctas < ctas) ctas = s->max_ctas;
    const S2dPlan plan = s2d_plan(box, g.batch, VN, K, (long long)ctas * WPC, a.dia_m, a.dia_n, a.dia_r);
    a.strip0 = plan.strip0; a.strips = plan.strips; a.segs = plan.segs; a.seg_len = plan.seg_len;
    a.row_lo = box.m_lo; a.row_hi = box.m_hi;
    a.units = (long long)g.batch * plan.segs * plan.strips;
    const long long need = (a.units + WPC - 1) / WPC;
    const unsigned grid = (unsigned)(need < ctas ? need : ctas);
    const size_t smem = stream2d_smem_bytes<R, K, RBL>();
    auto go = [&](auto kernel) -> int {
        QW_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kernel<<<grid, WPC * 32, smem, s->stream>>>(a);
        return QW_OK;
    };
    int rc = g.boundary == QW_OPEN ? go(step_stream2d_kernel<R, KIND, true, K, RBL>) : go(step_stream2d_kernel<R, KIND, false, K, RBL>);
    if (rc) return rc;
    QW_LAUNCH_CHECK(s, "step_stream2d_kernel");
    {   // site-steps actually computed: the valid outputs of the units the kernel's diamond test leaves active
        double sites = 0.0;
        for (int sg = 0; sg < plan.segs; ++sg) {
            const long long a0 = box.m_lo + sg * plan.seg_len, b0 = a0 + plan.seg_len <= box.m_hi + 1 ? a0 + plan.seg_len : box.m_hi + 1;
            if (a0 >= b0) continue;
            for (int st = 0; st < plan.strips; ++st) {
                const long long n_lo = (long long)(plan.strip0 + st) * VN;
                if (!s2d_unit_active(a0, b0, n_lo, n_lo + VN - 1, a.dia_m, a.dia_n, a.dia_r)) continue;
                const long long hn = n_lo + VN <= g.en ? VN : g.en - n_lo;
                if (hn > 0) sites += (double)(b0 - a0) * (double)hn;
            }
        }
        s->touched += sites * (double)g.batch * K;
    }
    return QW_OK;
}

// Instances: depths 2 .. 8 (2 .. 6 with link draws, which spill beyond), + 10 for complex64 without link draws.  (k = 12 was
// built and measured — never faster than k = 8 or 10, profiles/r02_stream2d.md — and dropped for its compile time.)
// Not static: the coins of one dtype are spread over two translation units (QW_S2D_EXTERN / QW_S2D_DEFINE below).
template <typename R, int KIND, bool RBL>
int s2d_launch_kind(qw_sim *s, int in_buf, int out_buf, int k, const Box &box) {
    switch (k) {
#ifndef QW_S2D_DEV                    // (tuning builds compile the deep float instances of one coin only)
        case 2: return s2d_launch_k<R, KIND, 2, RBL>(s, in_buf, out_buf, box);
        case 4: return s2d_launch_k<R, KIND, 4, RBL>(s, in_buf, out_buf, box);
        case 6: return s2d_launch_k<R, KIND, 6, RBL>(s, in_buf, out_buf, box);
#endif
        default: break;
    }
    if constexpr (!RBL) {
        if (k == 8) return s2d_launch_k<R, KIND, 8, RBL>(s, in_buf, out_buf, box);
        if constexpr (sizeof(R) == 4) {          // the deep pipeline: complex64 without link draws (stream2d_max_k)
            if (k == 10) return s2d_launch_k<R, KIND, 10, RBL>(s, in_buf, out_buf, box);
        }
    }
    return fail(QW_EINVAL, "streaming 2D step depth %d has no kernel instance here", k);
}
#define QW_S2D_EXTERN(R, KIND, RBL) extern template int s2d_launch_kind<R, KIND, RBL>(qw_sim *, int, int, int, const Box &);
#define QW_S2D_DEFINE(R, KIND, RBL) template int s2d_launch_kind<R, KIND, RBL>(qw_sim *, int, int, int, const Box &);

template <typename R, bool RBL>
static int s2d_launch(qw_sim *s, int in_buf, int out_buf, int k, const Box &box) {
    switch (s->coin_kind) {
#ifndef QW_S2D_DEV
        case COIN_GROVER4: return s2d_launch_kind<R, COIN_GROVER4, RBL>(s, in_buf, out_buf, k, box);
        case COIN_HXH4:    return s2d_launch_kind<R, COIN_HXH4, RBL>(s, in_buf, out_buf, k, box);
#endif
        case COIN_DFT4:    return s2d_launch_kind<R, COIN_DFT4, RBL>(s, in_buf, out_buf, k, box);
        default:           return s2d_launch_kind<R, COIN_GENERAL, RBL>(s, in_buf, out_buf, k, box);
    }
}

}  // namespace qw
