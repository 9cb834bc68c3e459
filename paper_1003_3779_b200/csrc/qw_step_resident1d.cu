// qw_step_resident1d.cu — SM-resident 1D walks: one CTA per walk keeps the whole state in registers
// for ALL n steps of a qw_step call, so HBM is touched only at the start and at the end
// (BASELINE.json:configs[0] and [4]).
//
// Thread `tid` owns the M consecutive sites tid*M .. tid*M+M-1 of both coin planes.  As in the
// temporally blocked kernel the shift of PAPER.md:46 eq. 3 is a renaming of registers inside a
// lane (at step s logical site i lives in Rp[(i - s) mod M], Lp[(i + s) mod M]); the one element per
// plane that crosses a lane boundary travels by warp shuffle, the one per warp that crosses a warp
// boundary through a double-buffered shared-memory slot (one __syncthreads per step).
// Per-walk coins C_w (the coin family may differ per walk) are read once into
// registers; per-site phases e^{i phi_x} (BASELINE.json:configs[4]) live in shared memory.
// Light cone: a warp whose 32*M sites cannot have been reached yet holds exact
// zeros and skips its coin arithmetic.
#include "qw_coin.cuh"

namespace qw {

// Launch shapes (sites per thread M, threads, CTAs per SM) are chosen in launch_resident_t: two CTAs per SM (the
// second one hides the first one's barrier) of up to 13 warps with M = 5 sites per thread for walks of up to 2080
// sites (BASELINE.json:configs[4]: 2049), M = 6 up to 2304, one CTA of 512 threads x 8 sites up to 4096.
constexpr int RES_MAX_SITES = 4096;

template <typename R>
struct Resident1dArgs {
    const typename Cx<R>::T *in;
    typename Cx<R>::T *out;
    long long n_sites, walk_stride, plane_stride;
    long long n_steps;
    long long x_off;                   // first site of thread 0: the CTA covers [x_off, x_off + threads * M) (a stage of the
                                       // light cone, see launch_resident_shape); everything outside is exactly zero
    const typename Cx<R>::T *coins;    // per-walk matrices or nullptr (uniform)
    const typename Cx<R>::T *phases;   // [walk][site] or nullptr
    int window;                        // 1: skip warps outside the light cone
    long long centre, radius0;
    R coin[8];
};

template <typename R>
struct ResidentCtx {
    typename Cx<R>::T *xR, *xL, *wrapR, *wrapL;         // exchange rows [2][T + 2] each (T = threads), wrap slots [2], [2]
    int xstride;                                        // T + 2
    const typename Cx<R>::T *ph;                        // padded per-site phases of this walk (shared)
    int lane, wid, nw, tid;
    bool lo_thread;        // owns site 0
    int hi_index;          // logical index of site N-1 inside this thread, or -1
    bool hi_warp;          // some lane of this warp owns site N-1
    long long warp_lo, warp_hi;   // first / last site of this warp's tile
    int window;
    long long centre, radius0;
};

template <typename R> __device__ __forceinline__ cplx<R> shfl_up_cx(cplx<R> v) {
    v.re = __shfl_up_sync(0xffffffffu, v.re, 1);
    v.im = __shfl_up_sync(0xffffffffu, v.im, 1);
    return v;
}
template <typename R> __device__ __forceinline__ cplx<R> shfl_down_cx(cplx<R> v) {
    v.re = __shfl_down_sync(0xffffffffu, v.re, 1);
    v.im = __shfl_down_sync(0xffffffffu, v.im, 1);
    return v;
}
template <typename R> __device__ __forceinline__ typename Cx<R>::T to_v(cplx<R> z) {
    typename Cx<R>::T v; v.x = z.re; v.y = z.im; return v;
}
template <typename R> __device__ __forceinline__ cplx<R> from_v(typename Cx<R>::T v) { return cplx<R>{v.x, v.y}; }

// One walk step; U = (steps done so far) mod M, s = steps done so far in this launch.
template <typename R, int M, int KIND, bool PHASES, bool OPEN, int U>
__device__ __forceinline__ void resident_step(cplx<R> (&Rp)[M], cplx<R> (&Lp)[M], const R *C,
                                              const ResidentCtx<R> &cx, long long s) {
    bool active = true;
    if (cx.window) {
        const long long r = cx.radius0 + s + 1;
        active = (cx.warp_lo <= cx.centre + r) && (cx.warp_hi >= cx.centre - r);
    }
    if (active) {
#pragma unroll
        for (int i = 0; i < M; ++i) {
            const int q = (i - U + M) % M, p = (i + U) % M;
            cplx<R> v[2] = {Rp[q], Lp[p]};
            apply_coin<R, 2, KIND>(C, v);
            if constexpr (PHASES) {
                const cplx<R> ph = from_v<R>(cx.ph[cx.tid * (M | 1) + i]);
                v[0] = cx_mul(ph.re, ph.im, v[0]);
                v[1] = cx_mul(ph.re, ph.im, v[1]);
            }
            Rp[q] = v[0];
            Lp[p] = v[1];
        }
    }
    constexpr int QS = (M - 1 - U + M) % M;   // phi_R of logical M-1 -> becomes R' of logical 0
    constexpr int PS = U % M;                 // phi_L of logical 0   -> becomes L' of logical M-1
    const cplx<R> outR = Rp[QS], outL = Lp[PS];
    cplx<R> hiR = {0, 0};                     // phi_R of site N-1 (needed by the wall / the wrap)
    if (cx.hi_warp) {
#pragma unroll
        for (int i = 0; i < M; ++i)
            if (i == cx.hi_index) hiR = Rp[(i - U + M) % M];
    }
    // The element per plane that leaves the thread goes through a shared-memory row (thread t writes entry t + 1, reads
    // entry t of the R row and entry t + 2 of the L row; entries 0 and T + 1 are zeros: beyond the CTA's range there is
    // nothing): two stores, the step's barrier, two loads — no shuffles, no special case at warp boundaries.  (An FP64
    // instruction holds the issue port for two cycles, so the 8 SHFL + ~12 register moves this replaces were paid in FP64 time.)
    const int par = (int)(s & 1);
    typename Cx<R>::T *xr = cx.xR + par * cx.xstride + cx.tid, *xl = cx.xL + par * cx.xstride + cx.tid;
    xr[1] = to_v<R>(outR);
    xl[1] = to_v<R>(outL);
    if constexpr (!OPEN) {
        if (cx.hi_index >= 0) cx.wrapR[par] = to_v<R>(hiR);
        if (cx.lo_thread) cx.wrapL[par] = to_v<R>(outL);
    }
    if (cx.nw > 1) __syncthreads(); else __syncwarp();
    Rp[QS] = from_v<R>(xr[0]);
    Lp[PS] = from_v<R>(xl[2]);
    // site 0 and site N-1: reflecting walls (RBL = 0) or the periodic seam
    if (cx.lo_thread) Rp[QS] = OPEN ? outL : from_v<R>(cx.wrapR[par]);
    if (cx.hi_warp) {
        const cplx<R> fix = OPEN ? hiR : from_v<R>(cx.wrapL[par]);
#pragma unroll
        for (int i = 0; i < M; ++i)
            if (i == cx.hi_index) Lp[(i + U + 1) % M] = fix;
    }
}

template <typename R, int M, int KIND, bool PHASES, bool OPEN, int U>
struct ResidentUnroll {
    static __device__ __forceinline__ void run(cplx<R> (&Rp)[M], cplx<R> (&Lp)[M], const R *C,
                                               const ResidentCtx<R> &cx, long long s, int count) {
        if (U < count) {
            resident_step<R, M, KIND, PHASES, OPEN, U>(Rp, Lp, C, cx, s + U);
            if constexpr (U + 1 < M) ResidentUnroll<R, M, KIND, PHASES, OPEN, U + 1>::run(Rp, Lp, C, cx, s, count);
        }
    }
};

template <typename R, int M, int KIND, bool PHASES, bool OPEN, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB)
step_resident1d_kernel(const Resident1dArgs<R> a) {
    typedef typename Cx<R>::T V;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, nw = blockDim.x >> 5;
    const long long w = blockIdx.x, N = a.n_sites;
    V *sm = reinterpret_cast<V *>(smem_raw);
    ResidentCtx<R> cx;
    const int T = blockDim.x;
    cx.xstride = T + 2;
    cx.xR = sm; cx.xL = sm + 2 * (T + 2); cx.wrapR = sm + 4 * (T + 2); cx.wrapL = sm + 4 * (T + 2) + 2;
    V *ph = sm + 4 * (T + 2) + 4;
    if (tid < 2) {                                  // the zero entries beyond both ends of the exchange rows
        V z; z.x = 0; z.y = 0;
        for (int par = 0; par < 2; ++par) {
            cx.xR[par * (T + 2) + tid * (T + 1)] = z;
            cx.xL[par * (T + 2) + tid * (T + 1)] = z;
        }
    }
    cx.ph = ph;
    cx.tid = tid; cx.lane = tid & 31; cx.wid = tid >> 5; cx.nw = nw;
    const long long x0 = a.x_off + (long long)tid * M;
    cx.lo_thread = (tid == 0) && a.x_off == 0;
    cx.hi_index = (N - 1 >= x0 && N - 1 < x0 + M) ? (int)(N - 1 - x0) : -1;
    cx.hi_warp = __any_sync(0xffffffffu, cx.hi_index >= 0);
    cx.warp_lo = a.x_off + (long long)cx.wid * 32 * M;
    cx.warp_hi = cx.warp_lo + 32 * M - 1;
    cx.window = a.window; cx.centre = a.centre; cx.radius0 = a.radius0;

    if constexpr (PHASES) {
        for (long long e = tid; e < (long long)blockDim.x * M; e += blockDim.x) {
            V z; z.x = 0; z.y = 0;
            if (a.x_off + e < N) z = a.phases[w * N + a.x_off + e];
            ph[(e / M) * (M | 1) + (e % M)] = z;       // odd row length: conflict-free 16-byte reads
        }
    }
    R C[8];
    if (a.coins) {
        const R *Cg = reinterpret_cast<const R *>(a.coins + w * 4);
#pragma unroll
        for (int i = 0; i < 8; ++i) C[i] = Cg[i];
    } else {
#pragma unroll
        for (int i = 0; i < 8; ++i) C[i] = a.coin[i];
    }
    cplx<R> Rp[M], Lp[M];
    const V *inw = a.in + w * a.walk_stride;
#pragma unroll
    for (int i = 0; i < M; ++i) {
        V r, l; r.x = r.y = 0; l.x = l.y = 0;
        if (x0 + i < N) { r = inw[x0 + i]; l = inw[a.plane_stride + x0 + i]; }
        Rp[i] = from_v<R>(r); Lp[i] = from_v<R>(l);
    }
    __syncthreads();

    long long s = 0;
    for (; s + M <= a.n_steps; s += M)
        ResidentUnroll<R, M, KIND, PHASES, OPEN, 0>::run(Rp, Lp, C, cx, s, M);
    const int rem = (int)(a.n_steps - s);
    if (rem > 0) {
        ResidentUnroll<R, M, KIND, PHASES, OPEN, 0>::run(Rp, Lp, C, cx, s, rem);
        // undo the register renaming of the last `rem` steps: logical i sits in Rp[(i-rem)%M], Lp[(i+rem)%M]
        for (int j = 0; j < rem; ++j) {
            const cplx<R> tr = Rp[M - 1], tl = Lp[0];
#pragma unroll
            for (int i = M - 1; i > 0; --i) Rp[i] = Rp[i - 1];
            Rp[0] = tr;
#pragma unroll
            for (int i = 0; i < M - 1; ++i) Lp[i] = Lp[i + 1];
            Lp[M - 1] = tl;
        }
    }
    V *outw = a.out + w * a.walk_stride;
#pragma unroll
    for (int i = 0; i < M; ++i) {
        if (x0 + i < N) { outw[x0 + i] = to_v<R>(Rp[i]); outw[a.plane_stride + x0 + i] = to_v<R>(Lp[i]); }
    }
}

bool resident1d_eligible(const qw_sim *s) {
    const Geom &g = s->g;
    return g.dim == 1 && g.en <= RES_MAX_SITES && s->coin_mode != QW_COIN_PER_SITE && !s->d_broken && !s->rbl &&
           g.batch <= 0x7fffffffLL;
}

// One launch = all walks advanced `steps` steps by CTAs of `threads` threads that cover the sites [x_off, x_off + threads*M).
template <typename R, int M, int KIND, bool PHASES, int MAXT, int MINB>
static int launch_resident_stage(qw_sim *s, const void *in, void *out, long long steps, long long x_off, int threads,
                                 long long radius0, bool cone_ok) {
    typedef typename Cx<R>::T V;
    const Geom &g = s->g;
    Resident1dArgs<R> a;
    a.in = static_cast<const V *>(in); a.out = static_cast<V *>(out);
    a.n_sites = g.en; a.walk_stride = g.walk_stride; a.plane_stride = g.plane_stride; a.n_steps = steps;
    a.x_off = x_off;
    a.coins = s->coin_mode == QW_COIN_PER_WALK ? static_cast<const V *>(s->d_coin) : nullptr;
    a.phases = static_cast<const V *>(s->d_phases);
    a.window = cone_ok ? 1 : 0; a.centre = s->centre[0]; a.radius0 = radius0;
    for (int i = 0; i < 8; ++i) a.coin[i] = (R)s->h_coin[i];
    const int nw = threads / 32;
    const size_t smem = sizeof(V) * (size_t)(4 * (threads + 2) + 4 + (PHASES ? (size_t)threads * (M | 1) : 0));
    auto launch = [&](auto kernel) -> int {
        if (smem > 48 * 1024)
            QW_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kernel<<<(unsigned)g.batch, threads, smem, s->stream>>>(a);
        return QW_OK;
    };
    int rc = g.boundary == QW_OPEN ? launch(step_resident1d_kernel<R, M, KIND, PHASES, true, MAXT, MINB>)
                                   : launch(step_resident1d_kernel<R, M, KIND, PHASES, false, MAXT, MINB>);
    if (rc) return rc;
    QW_LAUNCH_CHECK(s, "step_resident1d_kernel");
    {   // site-steps actually computed: the warps the per-step cone test of the kernel leaves active
        double touched = 0.0;
        for (long long st = 0; st < steps; ++st) {
            const long long r = radius0 + st + 1;
            for (int wi = 0; wi < nw; ++wi) {
                const long long lo = x_off + (long long)wi * 32 * M, hi = lo + 32 * M - 1;
                if (lo >= g.en) break;
                if (!a.window || (lo <= a.centre + r && hi >= a.centre - r)) touched += (double)((hi < g.en ? hi : g.en - 1) - lo + 1);
            }
        }
        s->touched += touched * (double)g.batch;
    }
    return QW_OK;
}

// n steps of all walks.  With a known light cone (after a delta start the walker is within t sites of its
// origin) the first steps need only the few warps around the origin: the run is cut into STAGES whose CTAs cover 2, 4, 8, ...
// warps' worth of sites around the cone (everything outside is exactly zero in both buffers) — small CTAs, many per SM —
// until the cone needs the whole walk.  A stage ends when the cone (+ M + 1 sites of margin, so that the end threads of the
// CTA hold nothing but zeros and need no boundary code) would leave its range; ranges are clamped to the lattice, a clamped
// side is a real wall.  Without a cone: one launch over the whole walk.
template <typename R, int M, int KIND, bool PHASES, int MAXT, int MINB>
static int launch_resident_shape(qw_sim *s, const void *in, void *out, long long n) {
    const Geom &g = s->g;
    int full_threads = (int)((g.en + M - 1) / M);
    full_threads = (full_threads + 31) / 32 * 32;
    // the cone test is only meaningful while the cone has not wrapped around a periodic lattice
    const bool cone_ok = s->window_enabled && s->window_valid &&
                         (g.boundary == QW_OPEN || (s->centre[0] - (s->radius + n + 1) >= 0 && s->centre[0] + (s->radius + n + 1) < g.en));
    struct Stage { long long steps, x_off; int threads; };
    Stage plan[12];
    int np = 0;
    long long done = 0, radius = s->radius;
    // (staging pays when there are enough walks to fill the machine with small CTAs; a single walk is latency bound)
    if (cone_ok && g.batch >= s->sm_count) {
        static const int widths[] = {2, 3, 4, 6, 8, 10, 12, 16, 24};
        for (int wi = 0; wi < 9 && np < 10 && done < n; ++wi) {
            const int nw = widths[wi];
            if (nw * 32 >= full_threads) break;
            const long long S = (long long)nw * 32 * M;
            long long lo = s->centre[0] - S / 2;
            if (lo < 0) lo = 0;
            if (lo + S > g.en) lo = g.en - S;
            if (lo < 0) break;
            lo = lo / 2 * 2;                                           // 16-byte aligned complex64 rows stay aligned
            // steps this range can hold: after t steps the support is within radius + t (+1 of pad) of the centre
            long long tmax = n - done;
            if (lo > 0) { const long long t = (s->centre[0] - lo) - (M + 1) - (radius + 1); if (t < tmax) tmax = t; }
            if (lo + S < g.en) { const long long t = (lo + S - 1 - s->centre[0]) - (M + 1) - (radius + 1); if (t < tmax) tmax = t; }
            if (tmax < 16) continue;
            plan[np++] = Stage{tmax, lo, nw * 32};
            done += tmax; radius += tmax;
        }
    }
    if (done < n) plan[np++] = Stage{n - done, 0, full_threads};
    if (np % 2 == 0) {       // an even number of launches would end in the input buffer: fold the first stage into the second
        plan[1].steps += plan[0].steps;
        for (int i = 0; i + 1 < np; ++i) plan[i] = plan[i + 1];
        --np;
    }
    const void *src = in;
    void *dst = out;
    radius = s->radius;
    for (int i = 0; i < np; ++i) {
        int rc = launch_resident_stage<R, M, KIND, PHASES, MAXT, MINB>(s, src, dst, plan[i].steps, plan[i].x_off, plan[i].threads,
                                                                      radius, cone_ok);
        if (rc) return rc;
        radius += plan[i].steps;
        const void *t = src; src = dst; dst = const_cast<void *>(t);
    }
    return QW_OK;
}

template <typename R, int KIND, bool PHASES>
static int launch_resident_t(qw_sim *s, const void *in, void *out, long long n) {
    const long long N = s->g.en;
    // measured on BASELINE.json:configs[4] (profiles/r01_blocked_resident.md, "launch shapes"): few sites per thread keep
    // the M-step unrolled body inside the 32 KB instruction cache and make the light-cone test (per warp) finer
    if (N <= 416 * 5) return launch_resident_shape<R, 5, KIND, PHASES, 416, 2>(s, in, out, n);
    if (N <= 384 * 6) return launch_resident_shape<R, 6, KIND, PHASES, 384, 2>(s, in, out, n);
    return launch_resident_shape<R, 8, KIND, PHASES, 512, 1>(s, in, out, n);
}

int launch_step_resident1d(qw_sim *s, const void *in, void *out, long long n) {
    const bool had = s->coin_mode == QW_COIN_UNIFORM && s->coin_kind == COIN_HADAMARD;
    const bool ph = s->d_phases != nullptr;
    if (s->dtype == QW_C128) {
        if (had) return ph ? launch_resident_t<double, COIN_HADAMARD, true>(s, in, out, n)
                           : launch_resident_t<double, COIN_HADAMARD, false>(s, in, out, n);
        return ph ? launch_resident_t<double, COIN_GENERAL, true>(s, in, out, n)
                  : launch_resident_t<double, COIN_GENERAL, false>(s, in, out, n);
    }
    if (had) return ph ? launch_resident_t<float, COIN_HADAMARD, true>(s, in, out, n)
                       : launch_resident_t<float, COIN_HADAMARD, false>(s, in, out, n);
    return ph ? launch_resident_t<float, COIN_GENERAL, true>(s, in, out, n)
              : launch_resident_t<float, COIN_GENERAL, false>(s, in, out, n);
}

}  // namespace qw
