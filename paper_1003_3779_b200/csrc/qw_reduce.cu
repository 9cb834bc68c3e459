// qw_reduce.cu — the per-vertex probability distribution P(x) = sum_coin |alpha|^2
// (Figs. 3-4) and its moments (norm of PAPER.md:56 eq. 4 / :78 eq. 6; mean and
// variance as BASELINE.json:north_star asks).  Both are one streaming pass over the state planes with
// 128-bit loads: HBM-bound.  Moments: per-thread FP64 accumulation about a LOCAL reference point, warp
// shuffles, a shared-memory tree per block, and a second, atomic-free pass over the block partials that
// shifts every partial to the global mean (no E[x^2] - E[x]^2 cancellation), so the result is
// deterministic and accurate for narrow distributions far from the lattice centre.
#include "qw_coin.cuh"

namespace qw {

constexpr int RED_BLOCK = 256;

// |z|^2 summed over the CD planes for VEC consecutive sites starting at element index idx (16-byte aligned loads).
// Accumulated in the type of the output: R for qw_probabilities, double for the moments.
template <typename R, typename ACC, int CD, int VEC>
__device__ __forceinline__ void site_probs(const typename Cx<R>::T *__restrict__ st, long long plane_stride, long long idx,
                                           ACC (&p)[VEC]) {
#pragma unroll
    for (int v = 0; v < VEC; ++v) p[v] = 0;
#pragma unroll
    for (int c = 0; c < CD; ++c) {
        const typename Cx<R>::T *src = st + c * plane_stride + idx;
        if constexpr (sizeof(R) == 8) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                const double2 z = __ldcs(src + v);              // streaming: every amplitude is read exactly once
                p[v] = fma((ACC)z.x, (ACC)z.x, p[v]);
                p[v] = fma((ACC)z.y, (ACC)z.y, p[v]);
            }
        } else {
#pragma unroll
            for (int v = 0; v < VEC; v += 2) {
                const float4 z = __ldcs(reinterpret_cast<const float4 *>(src + v));
                p[v] = fma((ACC)z.x, (ACC)z.x, p[v]);
                p[v] = fma((ACC)z.y, (ACC)z.y, p[v]);
                p[v + 1] = fma((ACC)z.z, (ACC)z.z, p[v + 1]);
                p[v + 1] = fma((ACC)z.w, (ACC)z.w, p[v + 1]);
            }
        }
    }
}
template <typename R, typename ACC, int CD>
__device__ __forceinline__ ACC site_prob1(const typename Cx<R>::T *__restrict__ st, long long plane_stride, long long idx) {
    ACC p = 0;
#pragma unroll
    for (int c = 0; c < CD; ++c) {
        const typename Cx<R>::T z = st[c * plane_stride + idx];
        p = fma((ACC)z.x, (ACC)z.x, p);
        p = fma((ACC)z.y, (ACC)z.y, p);
    }
    return p;
}

// sites per thread: two 16-byte loads per plane in flight (complex128: 2 sites, complex64: 4 sites)
template <typename R> struct RedVec { static constexpr int value = sizeof(R) == 8 ? 2 : 4; };

template <typename R, int CD>
__global__ void __launch_bounds__(RED_BLOCK)
prob_kernel(const typename Cx<R>::T *__restrict__ st, R *__restrict__ out, long long em, long long en, long long pitch,
            long long walk_stride, long long plane_stride, int chunks_per_row) {
    constexpr int VEC = RedVec<R>::value;
    const long long blk = blockIdx.x;
    const long long rowid = blk / chunks_per_row;               // walk * em + m
    const long long n = ((blk - rowid * chunks_per_row) * RED_BLOCK + threadIdx.x) * VEC;
    if (n >= en) return;
    const long long w = rowid / em, m = rowid - w * em;
    const long long idx = w * walk_stride + m * pitch + n;
    R *o = out + rowid * en + n;
    if (n + VEC <= en) {
        R p[VEC];
        site_probs<R, R, CD, VEC>(st, plane_stride, idx, p);
        if ((reinterpret_cast<uintptr_t>(o) & 15) == 0) {       // rows of odd length: not every row start is 16-byte aligned
            if constexpr (sizeof(R) == 8) *reinterpret_cast<double2 *>(o) = make_double2(p[0], p[1]);
            else *reinterpret_cast<float4 *>(o) = make_float4(p[0], p[1], p[2], p[3]);
        } else {
#pragma unroll
            for (int v = 0; v < VEC; ++v) o[v] = p[v];
        }
    } else {
        for (int v = 0; n + v < en; ++v) o[v] = site_prob1<R, R, CD>(st, plane_stride, idx + v);
    }
}

template <typename R, int CD>
static int launch_prob_t(qw_sim *s, const void *state, void *out) {
    const Geom &g = s->g;
    constexpr int PER_BLOCK = RED_BLOCK * RedVec<R>::value;
    const int cpr = (int)((g.en + PER_BLOCK - 1) / PER_BLOCK);
    const long long blocks = g.batch * g.em * cpr;
    if (blocks > 0x7fffffffLL) return fail(QW_EUNSUPPORTED, "lattice too large for one launch");
    prob_kernel<R, CD><<<(unsigned)blocks, RED_BLOCK, 0, s->stream>>>(
        static_cast<const typename Cx<R>::T *>(state), static_cast<R *>(out), g.em, g.en, g.pitch, g.walk_stride,
        g.plane_stride, cpr);
    QW_LAUNCH_CHECK(s, "prob_kernel");
    return QW_OK;
}

// Ensemble average over the batch axis: Pbar(x) = (1/B) sum_w P_w(x) (the averaged distribution of the random-broken-links
// model: every walk of a batch draws its own links).  One thread takes VEC consecutive sites of a lattice
// row and runs over the walks in order (FP64 accumulation: deterministic, and the mean of complex64 walks loses nothing).
template <typename R, int CD>
__global__ void __launch_bounds__(RED_BLOCK)
prob_mean_kernel(const typename Cx<R>::T *__restrict__ st, R *__restrict__ out, long long batch, long long em, long long en,
                 long long pitch, long long walk_stride, long long plane_stride, int chunks_per_row) {
    constexpr int VEC = RedVec<R>::value;
    const long long blk = blockIdx.x;
    const long long m = blk / chunks_per_row;
    const long long n = ((blk - m * chunks_per_row) * RED_BLOCK + threadIdx.x) * VEC;
    if (n >= en) return;
    const double inv = 1.0 / (double)batch;
    R *o = out + m * en + n;
    if (n + VEC <= en) {
        double acc[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) acc[v] = 0.0;
        for (long long w = 0; w < batch; ++w) {
            double p[VEC];
            site_probs<R, double, CD, VEC>(st, plane_stride, w * walk_stride + m * pitch + n, p);
#pragma unroll
            for (int v = 0; v < VEC; ++v) acc[v] += p[v];
        }
#pragma unroll
        for (int v = 0; v < VEC; ++v) o[v] = (R)(acc[v] * inv);
    } else {
        for (int v = 0; n + v < en; ++v) {
            double acc = 0.0;
            for (long long w = 0; w < batch; ++w) acc += site_prob1<R, double, CD>(st, plane_stride, w * walk_stride + m * pitch + n + v);
            o[v] = (R)(acc * inv);
        }
    }
}

template <typename R, int CD>
static int launch_prob_mean_t(qw_sim *s, const void *state, void *out) {
    const Geom &g = s->g;
    constexpr int PER_BLOCK = RED_BLOCK * RedVec<R>::value;
    const int cpr = (int)((g.en + PER_BLOCK - 1) / PER_BLOCK);
    const long long blocks = g.em * cpr;
    if (blocks > 0x7fffffffLL) return fail(QW_EUNSUPPORTED, "lattice too large for one launch");
    prob_mean_kernel<R, CD><<<(unsigned)blocks, RED_BLOCK, 0, s->stream>>>(
        static_cast<const typename Cx<R>::T *>(state), static_cast<R *>(out), g.batch, g.em, g.en, g.pitch, g.walk_stride,
        g.plane_stride, cpr);
    QW_LAUNCH_CHECK(s, "prob_mean_kernel");
    return QW_OK;
}

int launch_probabilities_mean(qw_sim *s, const void *state, void *out) {
    if (s->dtype == QW_C128)
        return s->g.cdim == 2 ? launch_prob_mean_t<double, 2>(s, state, out) : launch_prob_mean_t<double, 4>(s, state, out);
    return s->g.cdim == 2 ? launch_prob_mean_t<float, 2>(s, state, out) : launch_prob_mean_t<float, 4>(s, state, out);
}

int launch_probabilities(qw_sim *s, const void *state, void *out) {
    if (s->dtype == QW_C128)
        return s->g.cdim == 2 ? launch_prob_t<double, 2>(s, state, out) : launch_prob_t<double, 4>(s, state, out);
    return s->g.cdim == 2 ? launch_prob_t<float, 2>(s, state, out) : launch_prob_t<float, 4>(s, state, out);
}

// ---- moments -----------------------------------------------------------------------------------
// Block partials, per (walk, block): the reference point (rm, rn) in lattice-centred coordinates and the raw sums ABOUT it:
// S0 = sum P, Sm = sum (xm - rm) P, Sn = sum (xn - rn) P, Smm, Snn, Smn.
constexpr int NPART = 8;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// A block owns a CONTIGUOUS range of work items; an item is one chunk of RED_BLOCK * VEC sites of one lattice row.
// Row and chunk come from one division per ITEM (not per site); inside an item every thread takes VEC consecutive sites.
template <typename R, int CD>
__global__ void __launch_bounds__(RED_BLOCK)
moments_partial_kernel(const typename Cx<R>::T *__restrict__ st, double *__restrict__ partials, long long em, long long en,
                       long long pitch, long long walk_stride, long long plane_stride, int blocks_per_walk,
                       long long items_per_block, int chunks_per_row) {
    constexpr int VEC = RedVec<R>::value;
    const long long w = blockIdx.x / blocks_per_walk;
    const int b = (int)(blockIdx.x - w * blocks_per_walk);
    const long long items = em * chunks_per_row;
    const long long it0 = (long long)b * items_per_block;
    const long long it1 = it0 + items_per_block < items ? it0 + items_per_block : items;
    const long long cm = em / 2, cn = en / 2;
    // reference point of the block: its first site
    const long long m_ref = it0 / chunks_per_row, n_ref = (it0 - m_ref * chunks_per_row) * (RED_BLOCK * VEC);
    double a0 = 0, am = 0, an = 0, amm = 0, ann = 0, amn = 0;
#pragma unroll 2
    for (long long it = it0; it < it1; ++it) {
        const long long m = it / chunks_per_row;
        const long long n = ((it - m * chunks_per_row) * RED_BLOCK + threadIdx.x) * VEC;
        if (n >= en) continue;
        const long long idx = w * walk_stride + m * pitch + n;
        double p[VEC];
        int nv = VEC;
        if (n + VEC <= en) {
            site_probs<R, double, CD, VEC>(st, plane_stride, idx, p);
        } else {
            nv = (int)(en - n);
#pragma unroll
            for (int v = 0; v < VEC; ++v) p[v] = v < nv ? site_prob1<R, double, CD>(st, plane_stride, idx + v) : 0.0;
        }
        const double dm = (double)(m - m_ref), dn0 = (double)(n - n_ref);
        double s0 = 0, s1 = 0, s2 = 0;
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            const double dn = dn0 + v;
            s0 += p[v];
            s1 = fma(dn, p[v], s1);
            s2 = fma(dn * dn, p[v], s2);
        }
        a0 += s0; an += s1; ann += s2;
        am = fma(dm, s0, am); amm = fma(dm * dm, s0, amm); amn = fma(dm, s1, amn);
    }
    __shared__ double sm[6][RED_BLOCK / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double acc[6] = {a0, am, an, amm, ann, amn};
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const double v = warp_sum(acc[k]);
        if (lane == 0) sm[k][wid] = v;
    }
    __syncthreads();
    if (wid == 0) {
        double *out = partials + (size_t)blockIdx.x * NPART;
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            double v = (lane < RED_BLOCK / 32) ? sm[k][lane] : 0.0;
            v = warp_sum(v);
            if (lane == 0) out[2 + k] = v;
        }
        if (lane == 0) { out[0] = (double)(m_ref - cm); out[1] = (double)(n_ref - cn); }
    }
}

// One warp per walk: pass 1 folds the block partials (fixed order) into the norm and the means, pass 2 shifts every
// partial to the mean and folds the central second moments.  A walk whose norm is exactly 0 reports all zeros.
__global__ void moments_final_kernel(const double *__restrict__ partials, double *__restrict__ out,
                                     long long batch, int blocks_per_walk, int dim) {
    const long long w = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (w >= batch) return;
    const double *P = partials + (size_t)w * blocks_per_walk * NPART;
    double s0 = 0, sm = 0, sn = 0;
    for (int b = lane; b < blocks_per_walk; b += 32) {
        const double *q = P + (size_t)b * NPART;
        s0 += q[2];
        sm += fma(q[0], q[2], q[3]);
        sn += fma(q[1], q[2], q[4]);
    }
    s0 = warp_sum(s0); sm = warp_sum(sm); sn = warp_sum(sn);
    const bool empty = !(s0 != 0.0);
    const double mm = empty ? 0.0 : sm / s0, mn = empty ? 0.0 : sn / s0;
    double cmm = 0, cnn = 0, cmn = 0;
    for (int b = lane; b < blocks_per_walk; b += 32) {
        const double *q = P + (size_t)b * NPART;
        const double dm = q[0] - mm, dn = q[1] - mn;          // block reference relative to the mean
        cmm += q[5] + 2.0 * dm * q[3] + dm * dm * q[2];
        cnn += q[6] + 2.0 * dn * q[4] + dn * dn * q[2];
        cmn += q[7] + dm * q[4] + dn * q[3] + dm * dn * q[2];
    }
    cmm = warp_sum(cmm); cnn = warp_sum(cnn); cmn = warp_sum(cmn);
    if (lane == 0) {
        const double inv = empty ? 0.0 : 1.0 / s0;
        if (dim == 1) {
            out[w * 3 + 0] = s0;
            out[w * 3 + 1] = mn;
            out[w * 3 + 2] = cnn * inv;
        } else {
            out[w * 6 + 0] = s0;
            out[w * 6 + 1] = mm;
            out[w * 6 + 2] = mn;
            out[w * 6 + 3] = cmm * inv;
            out[w * 6 + 4] = cnn * inv;
            out[w * 6 + 5] = cmn * inv;
        }
    }
}

template <typename R, int CD>
static void launch_mom_t(qw_sim *s, const void *state, unsigned grid, int bpw, long long ipb, int cpr) {
    const Geom &g = s->g;
    moments_partial_kernel<R, CD><<<grid, RED_BLOCK, 0, s->stream>>>(
        static_cast<const typename Cx<R>::T *>(state), s->partials, g.em, g.en, g.pitch, g.walk_stride, g.plane_stride, bpw,
        ipb, cpr);
}

int launch_moments(qw_sim *s, const void *state, double *out) {
    const Geom &g = s->g;
    const int vec = s->dtype == QW_C128 ? RedVec<double>::value : RedVec<float>::value;
    const int cpr = (int)((g.en + (long long)RED_BLOCK * vec - 1) / ((long long)RED_BLOCK * vec));
    const long long items = g.em * cpr;
    // enough blocks to fill the machine (16 CTAs of 256 threads per SM and a few waves), never more than the work
    long long bpw = (long long)s->sm_count * 32 / g.batch;
    if (bpw < 1) bpw = 1;
    if (bpw > items) bpw = items;
    const long long ipb = (items + bpw - 1) / bpw;
    bpw = (items + ipb - 1) / ipb;
    const long long blocks = bpw * g.batch;
    if (blocks > 0x7fffffffLL) return fail(QW_EUNSUPPORTED, "batch too large for one launch");
    const size_t need = (size_t)blocks * NPART;
    if (need > s->partials_count) {
        if (s->partials) { cudaStreamSynchronize(s->stream); cudaFree(s->partials); }
        s->partials = nullptr; s->partials_count = 0;
        QW_CUDA(cudaMalloc(&s->partials, need * sizeof(double)));
        s->partials_count = need;
    }
    if (s->dtype == QW_C128) { if (g.cdim == 2) launch_mom_t<double, 2>(s, state, (unsigned)blocks, (int)bpw, ipb, cpr); else launch_mom_t<double, 4>(s, state, (unsigned)blocks, (int)bpw, ipb, cpr); }
    else                     { if (g.cdim == 2) launch_mom_t<float, 2>(s, state, (unsigned)blocks, (int)bpw, ipb, cpr);  else launch_mom_t<float, 4>(s, state, (unsigned)blocks, (int)bpw, ipb, cpr); }
    QW_LAUNCH_CHECK(s, "moments_partial_kernel");
    const int warps = 4;
    moments_final_kernel<<<(unsigned)((g.batch + warps - 1) / warps), warps * 32, 0, s->stream>>>(
        s->partials, out, g.batch, (int)bpw, g.dim);
    QW_LAUNCH_CHECK(s, "moments_final_kernel");
    return QW_OK;
}

// ---- moments without any allocation (qw_moments_static) --------------------------------------------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
// the same two kernels as launch_moments, with the block partials in a file-scope device array of a fixed, modest size
// instead of the handle's lazily grown cudaMalloc buffer.  Every GPU that loads the library holds the array
// (QW_STATIC_PARTIAL_BLOCKS * NPART doubles = 512 KiB) until exit.  ALL calls on a device share it: every call overwrites
// all NPART entries of every block it uses before the second kernel reads them (nothing has to start at zero, nothing is
// accumulated across calls), so calls in ONE stream are safe one after the other, while calls that overlap on the GPU
// (different streams or handles at the same time) race.
constexpr long long QW_STATIC_PARTIAL_BLOCKS = 8192;
static __device__ __align__(256) double qw_static_partials[QW_STATIC_PARTIAL_BLOCKS * NPART];

// In host code the array's name is a host-side stand-in, not a device address: its device address is looked up once per
// device, with that device current, and that pointer is what the kernels get.
static double *static_partials_ptr(int device) {
    constexpr int MAXDEV = 64;
    static double *ptr[MAXDEV] = {};
    if (device < 0 || device >= MAXDEV) return nullptr;
    if (!ptr[device]) {
        double *p = nullptr;
        if (cudaGetSymbolAddress((void **)&p, qw_static_partials) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        ptr[device] = p;
    }
    return ptr[device];
}

template <typename R, int CD>
static void launch_mom_static_t(qw_sim *s, const void *state, double *partials, unsigned grid, int bpw, long long ipb, int cpr) {
    const Geom &g = s->g;
    moments_partial_kernel<R, CD><<<grid, RED_BLOCK, 0, s->stream>>>(
        static_cast<const typename Cx<R>::T *>(state), partials, g.em, g.en, g.pitch, g.walk_stride, g.plane_stride, bpw, ipb, cpr);
}

// out: DEVICE pointer.  The caller (qw_moments_static) has made s->device the current device.
int launch_moments_static(qw_sim *s, const void *state, double *out) {
    const Geom &g = s->g;
    if (g.batch > QW_STATIC_PARTIAL_BLOCKS)
        return fail(QW_EUNSUPPORTED, "qw_moments_static holds the partial sums of at most %lld blocks: batch %lld is too large "
                                     "(use qw_moments, which allocates)", QW_STATIC_PARTIAL_BLOCKS, g.batch);
    const int vec = s->dtype == QW_C128 ? RedVec<double>::value : RedVec<float>::value;
    const int cpr = (int)((g.en + (long long)RED_BLOCK * vec - 1) / ((long long)RED_BLOCK * vec));
    const long long items = g.em * cpr;
    // as launch_moments, with the blocks per walk capped by what the static array holds
    long long bpw = (long long)s->sm_count * 32 / g.batch;
    if (bpw > QW_STATIC_PARTIAL_BLOCKS / g.batch) bpw = QW_STATIC_PARTIAL_BLOCKS / g.batch;
    if (bpw < 1) bpw = 1;
    if (bpw > items) bpw = items;
    const long long ipb = (items + bpw - 1) / bpw;
    bpw = (items + ipb - 1) / ipb;
    const long long blocks = bpw * g.batch;
    if (blocks > QW_STATIC_PARTIAL_BLOCKS) return fail(QW_EUNSUPPORTED, "qw_moments_static: %lld blocks exceed the static scratch", blocks);
    double *partials = static_partials_ptr(s->device);
    if (!partials) return fail(QW_ECUDA, "cudaGetSymbolAddress(qw_static_partials) failed on device %d", s->device);
    if (s->dtype == QW_C128) { if (g.cdim == 2) launch_mom_static_t<double, 2>(s, state, partials, (unsigned)blocks, (int)bpw, ipb, cpr); else launch_mom_static_t<double, 4>(s, state, partials, (unsigned)blocks, (int)bpw, ipb, cpr); }
    else                     { if (g.cdim == 2) launch_mom_static_t<float, 2>(s, state, partials, (unsigned)blocks, (int)bpw, ipb, cpr);  else launch_mom_static_t<float, 4>(s, state, partials, (unsigned)blocks, (int)bpw, ipb, cpr); }
    QW_LAUNCH_CHECK(s, "moments_partial_kernel");
    const int warps = 4;
    moments_final_kernel<<<(unsigned)((g.batch + warps - 1) / warps), warps * 32, 0, s->stream>>>(partials, out, g.batch, (int)bpw, g.dim);
    QW_LAUNCH_CHECK(s, "moments_final_kernel");
    return QW_OK;
}

}  // namespace qw
