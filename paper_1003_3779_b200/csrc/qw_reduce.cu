// qw_reduce.cu — the per-vertex probability distribution P(x) = sum_coin |alpha|^2
// (Figs. 3-4) and its moments (norm of PAPER.md:56 eq. 4 / :78 eq. 6; mean and
// variance as BASELINE.json:north_star asks): per-thread FP64 accumulation, warp shuffles, a
// shared-memory tree per block, and a second, atomic-free pass over the block partials, so the
// result is deterministic.
#include "qw_coin.cuh"

namespace qw {

constexpr int RED_BLOCK = 256;

template <typename R, int CD>
__global__ void __launch_bounds__(RED_BLOCK)
prob_kernel(const typename Cx<R>::T *__restrict__ st, R *__restrict__ out, long long rows, long long em,
            long long en, long long pitch, long long walk_stride, long long plane_stride, int chunks_per_row) {
    const long long blk = blockIdx.x;
    const long long rowid = blk / chunks_per_row;               // walk * em + m
    const long long n = (blk - rowid * chunks_per_row) * RED_BLOCK + threadIdx.x;
    if (n >= en) return;
    const long long w = rowid / em, m = rowid - w * em;
    const long long idx = w * walk_stride + m * pitch + n;
    R p = 0;
#pragma unroll
    for (int c = 0; c < CD; ++c) {
        const typename Cx<R>::T z = st[c * plane_stride + idx];
        p = fma_rn(z.x, z.x, p);
        p = fma_rn(z.y, z.y, p);
    }
    out[rowid * en + n] = p;
}

template <typename R, int CD>
static int launch_prob_t(qw_sim *s, const void *state, void *out) {
    const Geom &g = s->g;
    const int cpr = (int)((g.en + RED_BLOCK - 1) / RED_BLOCK);
    const long long blocks = g.batch * g.em * cpr;
    if (blocks > 0x7fffffffLL) return fail(QW_EUNSUPPORTED, "lattice too large for one launch");
    prob_kernel<R, CD><<<(unsigned)blocks, RED_BLOCK, 0, s->stream>>>(
        static_cast<const typename Cx<R>::T *>(state), static_cast<R *>(out), g.batch * g.em, g.em, g.en,
        g.pitch, g.walk_stride, g.plane_stride, cpr);
    QW_LAUNCH_CHECK(s, "prob_kernel");
    return QW_OK;
}

int launch_probabilities(qw_sim *s, const void *state, void *out) {
    if (s->dtype == QW_C128)
        return s->g.cdim == 2 ? launch_prob_t<double, 2>(s, state, out) : launch_prob_t<double, 4>(s, state, out);
    return s->g.cdim == 2 ? launch_prob_t<float, 2>(s, state, out) : launch_prob_t<float, 4>(s, state, out);
}

// ---- moments -----------------------------------------------------------------------------------
// Raw sums per walk: S0 = sum P, Sm = sum xm P, Sn = sum xn P, Smm, Snn, Smn  (1D uses S0, Sn, Snn).
constexpr int NMOM = 6;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <typename R, int CD>
__global__ void __launch_bounds__(RED_BLOCK)
moments_partial_kernel(const typename Cx<R>::T *__restrict__ st, double *__restrict__ partials, long long em,
                       long long en, long long pitch, long long walk_stride, long long plane_stride,
                       int blocks_per_walk) {
    const long long w = blockIdx.y;
    const long long cm = em / 2, cn = en / 2;
    const long long sites = em * en;
    double acc[NMOM] = {0, 0, 0, 0, 0, 0};
    for (long long x = (long long)blockIdx.x * RED_BLOCK + threadIdx.x; x < sites;
         x += (long long)blocks_per_walk * RED_BLOCK) {
        const long long m = x / en, n = x - m * en;
        const long long idx = w * walk_stride + m * pitch + n;
        double p = 0.0;
#pragma unroll
        for (int c = 0; c < CD; ++c) {
            const typename Cx<R>::T z = st[c * plane_stride + idx];
            const double re = (double)z.x, im = (double)z.y;
            p = fma(re, re, p);
            p = fma(im, im, p);
        }
        const double xm = (double)(m - cm), xn = (double)(n - cn);
        acc[0] += p;
        acc[1] += xm * p;
        acc[2] += xn * p;
        acc[3] += xm * xm * p;
        acc[4] += xn * xn * p;
        acc[5] += xm * xn * p;
    }
    __shared__ double sm[NMOM][RED_BLOCK / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NMOM; ++k) {
        const double v = warp_sum(acc[k]);
        if (lane == 0) sm[k][wid] = v;
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int k = 0; k < NMOM; ++k) {
            double v = (lane < RED_BLOCK / 32) ? sm[k][lane] : 0.0;
            v = warp_sum(v);
            if (lane == 0) partials[(w * blocks_per_walk + blockIdx.x) * NMOM + k] = v;
        }
    }
}

// One warp per walk folds the block partials in a fixed order and forms the normalised moments.
__global__ void moments_final_kernel(const double *__restrict__ partials, double *__restrict__ out,
                                     long long batch, int blocks_per_walk, int dim) {
    const long long w = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (w >= batch) return;
    double acc[NMOM] = {0, 0, 0, 0, 0, 0};
    for (int b = lane; b < blocks_per_walk; b += 32)
#pragma unroll
        for (int k = 0; k < NMOM; ++k) acc[k] += partials[(w * blocks_per_walk + b) * NMOM + k];
#pragma unroll
    for (int k = 0; k < NMOM; ++k) acc[k] = warp_sum(acc[k]);
    if (lane == 0) {
        const double s0 = acc[0];
        const double mm = acc[1] / s0, mn = acc[2] / s0;
        if (dim == 1) {
            out[w * 3 + 0] = s0;
            out[w * 3 + 1] = mn;
            out[w * 3 + 2] = acc[4] / s0 - mn * mn;
        } else {
            out[w * 6 + 0] = s0;
            out[w * 6 + 1] = mm;
            out[w * 6 + 2] = mn;
            out[w * 6 + 3] = acc[3] / s0 - mm * mm;
            out[w * 6 + 4] = acc[4] / s0 - mn * mn;
            out[w * 6 + 5] = acc[5] / s0 - mm * mn;
        }
    }
}

int launch_moments(qw_sim *s, const void *state, double *out) {
    const Geom &g = s->g;
    // enough blocks to fill the machine, never more than the work
    long long want = (g.sites + (long long)RED_BLOCK * 8 - 1) / ((long long)RED_BLOCK * 8);
    long long cap = (long long)s->sm_count * 8 / (g.batch < 1 ? 1 : g.batch);
    if (cap < 1) cap = 1;
    if (want > cap) want = cap;
    if (want < 1) want = 1;
    const int bpw = (int)want;
    if (g.batch > 65535) return fail(QW_EUNSUPPORTED, "batch larger than 65535 walks");
    const size_t need = (size_t)g.batch * bpw * NMOM;
    if (need > s->partials_count) {
        if (s->partials) cudaFree(s->partials);
        s->partials = nullptr; s->partials_count = 0;
        QW_CUDA(cudaMalloc(&s->partials, need * sizeof(double)));
        s->partials_count = need;
    }
    dim3 grid((unsigned)bpw, (unsigned)g.batch);
#define QW_MOM(R, CD)                                                                                   \
    moments_partial_kernel<R, CD><<<grid, RED_BLOCK, 0, s->stream>>>(                                   \
        static_cast<const Cx<R>::T *>(state), s->partials, g.em, g.en, g.pitch, g.walk_stride,          \
        g.plane_stride, bpw)
    if (s->dtype == QW_C128) { if (g.cdim == 2) QW_MOM(double, 2); else QW_MOM(double, 4); }
    else                     { if (g.cdim == 2) QW_MOM(float, 2);  else QW_MOM(float, 4); }
#undef QW_MOM
    QW_LAUNCH_CHECK(s, "moments_partial_kernel");
    const int warps = 4;
    moments_final_kernel<<<(unsigned)((g.batch + warps - 1) / warps), warps * 32, 0, s->stream>>>(
        s->partials, out, g.batch, bpw, g.dim);
    QW_LAUNCH_CHECK(s, "moments_final_kernel");
    return QW_OK;
}

}  // namespace qw
