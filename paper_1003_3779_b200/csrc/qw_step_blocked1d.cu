// qw_step_blocked1d.cu — temporally blocked 1D step: k applications of U = S (I (x) C)
// (eq. 2) per HBM round trip, for a uniform coin on a 1D lattice.
//
// Design: every WARP owns an independent tile of 32*M
// consecutive sites: valid = 32*M - 2k output sites plus a k-site halo on each side (after k steps
// the influence of the unknown outside has travelled exactly k sites inwards).
// Lane j keeps the M consecutive sites j*M .. j*M+M-1 of both coin planes in registers.  One step:
//   coin    in place on every (R[i], L[i]) pair                           (eq. 1)
//   shift   R moves one site right, L one site left (eq. 3).  Inside a lane this is a RENAMING
//           of registers, not a move: at step s logical site i lives in Rp[(i - s) mod M] and
//           Lp[(i + s) mod M]; only the element that crosses the lane boundary moves, through
//           one warp shuffle per plane.  The step loop is unrolled M times so every register
//           index is a compile-time constant; k must be a multiple of M.
// No block-level synchronisation and no shared-memory traffic inside the k steps; shared memory
// is only the staging area that turns coalesced global accesses into lane-contiguous registers.
// Warps are persistent and prefetch their next tile with cp.async while the current one is advanced;
// the Hadamard coin runs with a deferred scale; open lattices align their first / last tile with the
// walls; a remainder of 4 .. 15 steps uses short M = 8 / M = 4 tiles (all explained where they occur).
// HBM bytes per site-step: coin_dim*sizeof(complex) * (32M/valid + 1) / k  instead of 2*coin_dim*sizeof(complex).
#include "qw_coin.cuh"

namespace qw {

constexpr int BLK1D_WARPS = 4;

template <typename R>
struct Blocked1dArgs {
    const typename Cx<R>::T *in;
    typename Cx<R>::T *out;
    long long n_sites;       // en
    long long walk_stride, plane_stride;
    long long tiles_per_walk, total_tiles;
    int k;                   // steps in this launch, multiple of M
    int valid;               // 32*M - 2k
    int boundary;
    R coin[8];
    R scale_m;               // deferred-scale Hadamard: s^M, applied once per M steps (see blocked1d_step)
};

template <typename R> __device__ __forceinline__ cplx<R> shfl_up1(cplx<R> v) {
    v.re = __shfl_up_sync(0xffffffffu, v.re, 1);
    v.im = __shfl_up_sync(0xffffffffu, v.im, 1);
    return v;
}
template <typename R> __device__ __forceinline__ cplx<R> shfl_down1(cplx<R> v) {
    v.re = __shfl_down_sync(0xffffffffu, v.re, 1);
    v.im = __shfl_down_sync(0xffffffffu, v.im, 1);
    return v;
}

// One walk step with s = U (mod M).
//
// Deferred scale (KIND == COIN_HADAMARD with M = 16; the short M = 8 / M = 4 tiles that mop up a remainder of 4 .. 15
// steps use the scaled evaluation of the fused kernel, bit for bit): the coin s*[[1,1],[1,-1]] is linear in s, so M consecutive steps equal
// M unscaled butterflies (phi_R = R + L, phi_L = R - L: 4 additions per site-step instead of 2 mul + 4 fma)
// followed by ONE multiplication by s^M.  Steps U = 0 .. M-2 run the bare butterfly, step U = M-1 runs the usual
// scaled evaluation with s^M (C[1], filled by the launcher) in place of s.  The intermediate values grow by at most
// 2^(M-1), far inside the exponent range, and are rescaled every M steps whatever the launch depth k, so the
// result does not depend on k.  It differs from M scaled single steps by rounding only (fewer roundings, in fact):
// <= 4 ulp per step (SURVEY.md 8(c) P13 "otherwise <= 4 ulp t").
template <typename R, int M, int KIND, bool OPEN, int U>
__device__ __forceinline__ void blocked1d_step(cplx<R> (&Rp)[M], cplx<R> (&Lp)[M], const R *C,
                                               int lane, int lo_lane, int hi_lane) {
#pragma unroll
    for (int i = 0; i < M; ++i) {
        const int q = (i - U + M) % M, p = (i + U) % M;
        cplx<R> v[2] = {Rp[q], Lp[p]};
        if constexpr (KIND == COIN_HADAMARD && M == 16) {
            if constexpr (U + 1 < M) {
                const cplx<R> r = v[0], l = v[1];
                v[0] = cx_add(r, l);
                v[1] = cx_sub(r, l);
            } else {
                apply_coin<R, 2, COIN_HADAMARD>(C + 1, v);      // C[1] = s^M
            }
        } else {
            apply_coin<R, 2, KIND>(C, v);
        }
        Rp[q] = v[0];
        Lp[p] = v[1];
    }
    constexpr int QS = (M - 1 - U + M) % M;     // holds phi_R of logical M-1, becomes R' of logical 0
    constexpr int PS = U % M;                   // holds phi_L of logical 0,   becomes L' of logical M-1
    if constexpr (OPEN) {
        // reflecting walls (PAPER.md:94-101 with RBL = 0): R'[0] = phi_L[0], L'[N-1] = phi_R[N-1].  The tiles are laid out
        // so that site 0 is always logical site 0 of lane lo_lane (first tile of a walk) and site N-1 logical site M-1 of
        // lane hi_lane (last tile, which ends exactly at the wall): the reflected value replaces what the shuffle brings.
        const cplx<R> outR = Rp[QS], outL = Lp[PS];
        Rp[QS] = shfl_up1(outR);
        Lp[PS] = shfl_down1(outL);
        if (lane == lo_lane) Rp[QS] = outL;
        if (lane == hi_lane) Lp[PS] = outR;
    } else {
        Rp[QS] = shfl_up1(Rp[QS]);
        Lp[PS] = shfl_down1(Lp[PS]);
    }
}

template <typename R, int M, int KIND, bool OPEN, int U>
struct Blocked1dUnroll {
    static __device__ __forceinline__ void run(cplx<R> (&Rp)[M], cplx<R> (&Lp)[M], const R *C, int lane, int lo_lane,
                                               int hi_lane) {
        blocked1d_step<R, M, KIND, OPEN, U>(Rp, Lp, C, lane, lo_lane, hi_lane);
        if constexpr (U + 1 < M) Blocked1dUnroll<R, M, KIND, OPEN, U + 1>::run(Rp, Lp, C, lane, lo_lane, hi_lane);
    }
};

// padded staging position of tile element e (row = owning lane): odd row length -> conflict-free
template <int M> __device__ __forceinline__ int stage_pos(int e) { return (e / M) * (M + 1) + (e % M); }

// 16- / 8-byte asynchronous global -> shared copy (LDGSTS); src_bytes = 0 writes zeros (sites outside an open lattice)
template <int BYTES>
__device__ __forceinline__ void cp_async_elem(void *smem_dst, const void *gmem_src, int src_bytes) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    if constexpr (BYTES == 16)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(gmem_src), "r"(src_bytes) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(d), "l"(gmem_src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// resident CTAs per SM the kernel is sized for: 2 x 4 warps for complex128 (3 staging planes of 8.5 KB per warp
// = 104 KB per CTA), 4 x 4 warps for complex64
template <typename R> struct Blocked1dMinBlocks { static constexpr int value = sizeof(R) == 8 ? 2 : 4; };

template <typename R, int M> constexpr size_t blocked1d_smem_bytes() {
    return (size_t)BLK1D_WARPS * 3 * 32 * (M + 1) * sizeof(typename Cx<R>::T);
}

// Persistent warps: warp g of the grid walks over tiles g, g + G, g + 2G, ...  While tile n is advanced k steps in
// registers, the input of tile n + G is already in flight (cp.async into the warp's two input planes of shared
// memory), so the HBM round trip of a tile hides behind the arithmetic of the previous one instead of adding to it
// (without the prefetch all resident warps load, compute and store in lock step: time = compute + memory).
template <typename R, int M, int KIND, bool OPEN>
__global__ void __launch_bounds__(BLK1D_WARPS * 32, Blocked1dMinBlocks<R>::value)
step_blocked1d_kernel(const Blocked1dArgs<R> a) {
    typedef typename Cx<R>::T V;
    constexpr int PLANE = 32 * (M + 1);
    extern __shared__ __align__(16) unsigned char blk1d_smem[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    V *st_in = reinterpret_cast<V *>(blk1d_smem) + (size_t)wid * 3 * PLANE;   // [2][PLANE]: prefetched input planes
    V *st_out = st_in + 2 * PLANE;                                            // [PLANE]: output staging
    const long long N = a.n_sites;
    const long long stride = (long long)gridDim.x * BLK1D_WARPS;
    long long tile_id = (long long)blockIdx.x * BLK1D_WARPS + wid;

    // tile id -> (walk, tile of the walk); total_tiles < 2^31 (checked by the launcher)
    auto split = [&](long long tid, long long &w, long long &t) {
        if (a.tiles_per_walk == a.total_tiles) { w = 0; t = tid; return; }
        const unsigned q = (unsigned)tid / (unsigned)a.tiles_per_walk;
        w = q; t = (long long)((unsigned)tid - q * (unsigned)a.tiles_per_walk);
    };
    // unwrapped coordinate of element 0 of tile t of a walk.  Open lattice: the LAST tile is shifted so that it ends exactly
    // at the wall (its outputs are the last `valid` sites; the tile before it stores only what lies in front of them)
    auto tile_start = [&](long long t) -> long long {
        if (OPEN && t == a.tiles_per_walk - 1) return N - a.valid - a.k;
        return t * a.valid - a.k;
    };
    // element i*32 + lane of a tile sits at stage_pos(lane) + i * STEP_I of a staging plane (M divides 32)
    constexpr int STEP_I = (32 / M) * (M + 1);
    const int pos_lane = stage_pos<M>(lane);

    // coalesced global -> padded shared, both planes of one tile, asynchronously
    auto prefetch = [&](long long tid) {
        long long w, t;
        split(tid, w, t);
        const long long start = tile_start(t);
        const V *inw = a.in + w * a.walk_stride;
        if (start >= 0 && start + 32 * M <= N) {             // interior tile: no wrap, no wall -> immediate offsets only
            const V *p0 = inw + start + lane, *p1 = p0 + a.plane_stride;
            V *d0 = st_in + pos_lane, *d1 = d0 + PLANE;
#pragma unroll
            for (int i = 0; i < M; ++i) cp_async_elem<(int)sizeof(V)>(d0 + i * STEP_I, p0 + i * 32, (int)sizeof(V));
#pragma unroll
            for (int i = 0; i < M; ++i) cp_async_elem<(int)sizeof(V)>(d1 + i * STEP_I, p1 + i * 32, (int)sizeof(V));
        } else {
#pragma unroll 1
            for (int plane = 0; plane < 2; ++plane) {
#pragma unroll 4
                for (int i = 0; i < M; ++i) {
                    long long x = start + i * 32 + lane;
                    bool ok = true;
                    if (OPEN) ok = (x >= 0) && (x < N);
                    else { if (x < 0) x += N; else if (x >= N) x -= N; }
                    cp_async_elem<(int)sizeof(V)>(st_in + plane * PLANE + pos_lane + i * STEP_I,
                                                  inw + plane * a.plane_stride + (ok ? x : 0), ok ? (int)sizeof(V) : 0);
                }
            }
        }
        cp_async_commit();
    };

    R C[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) C[i] = a.coin[i];
    if constexpr (KIND == COIN_HADAMARD && M == 16) C[1] = a.scale_m;   // the imaginary part of C[0][0] (zero) is not used

    if (tile_id < a.total_tiles) prefetch(tile_id);
    for (; tile_id < a.total_tiles; tile_id += stride) {
        long long w, t;
        split(tile_id, w, t);
        const long long start = tile_start(t);         // unwrapped coordinate of tile element 0
        V *outw = a.out + w * a.walk_stride;

        // ---- padded shared -> lane-contiguous registers
        cplx<R> Rp[M], Lp[M];
        cp_async_wait_all();
        __syncwarp();
#pragma unroll
        for (int i = 0; i < M; ++i) {
            const V zr = st_in[lane * (M + 1) + i], zl = st_in[PLANE + lane * (M + 1) + i];
            Rp[i] = cplx<R>{zr.x, zr.y};
            Lp[i] = cplx<R>{zl.x, zl.y};
        }
        __syncwarp();
        if (tile_id + stride < a.total_tiles) prefetch(tile_id + stride);

        // ---- k steps in registers
        int lo_lane = -1, hi_lane = -1;                // lanes that own site 0 (as logical site 0) / site N-1 (as logical M-1)
        if (OPEN) {
            if (t == 0) lo_lane = a.k / M;
            if (t == a.tiles_per_walk - 1) hi_lane = 31 - a.k / M;
        }
        for (int s = 0; s < a.k; s += M)
            Blocked1dUnroll<R, M, KIND, OPEN, 0>::run(Rp, Lp, C, lane, lo_lane, hi_lane);

        // ---- store the valid middle: registers -> padded shared -> coalesced global
        // sites this tile stores: [start + k, x_end).  Ring: the last tile is cut at N.  Open lattice: the tile before the
        // (shifted) last one is cut where the last one begins.
        const long long x_end_all = OPEN ? N - a.valid : N;
        const long long x_end = (OPEN && t == a.tiles_per_walk - 1) ? N : x_end_all;
        const bool whole = start + a.k + a.valid <= x_end;  // every valid output site of the tile is stored
        const int lk = lane - a.k;                          // element e = i*32 + lane is valid iff 0 <= e - k < valid
        V *o0 = outw + (start + a.k + lk);
#pragma unroll
        for (int plane = 0; plane < 2; ++plane) {
#pragma unroll
            for (int i = 0; i < M; ++i) {
                V z;
                if (plane == 0) { z.x = Rp[i].re; z.y = Rp[i].im; } else { z.x = Lp[i].re; z.y = Lp[i].im; }
                st_out[lane * (M + 1) + i] = z;
            }
            __syncwarp();
            V *op = o0 + plane * a.plane_stride;
            if (whole) {
#pragma unroll
                for (int i = 0; i < M; ++i)
                    if ((unsigned)(lk + i * 32) < (unsigned)a.valid) op[i * 32] = st_out[pos_lane + i * STEP_I];
            } else {
#pragma unroll 4
                for (int i = 0; i < M; ++i)
                    if ((unsigned)(lk + i * 32) < (unsigned)a.valid && start + a.k + lk + i * 32 < x_end)
                        op[i * 32] = st_out[pos_lane + i * STEP_I];
            }
            __syncwarp();
        }
    }
}

template <typename R, int M, int KIND, bool OPEN>
static int launch_blocked1d_k(qw_sim *s, const Blocked1dArgs<R> &a) {
    auto kern = step_blocked1d_kernel<R, M, KIND, OPEN>;
    constexpr size_t smem = blocked1d_smem_bytes<R, M>();
    static int ctas_per_sm_dev[64];  // per instantiation AND per device: the function attribute is a per-device setting
    int &ctas_per_sm = ctas_per_sm_dev[s->device & 63];
    if (ctas_per_sm == 0) {
        QW_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int n = 0;
        QW_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, BLK1D_WARPS * 32, smem));
        if (n < 1) return fail(QW_ECUDA, "step_blocked1d_kernel does not fit on an SM (%zu bytes of shared memory)", smem);
        ctas_per_sm = n;
    }
    if (a.total_tiles > 0x7fffffffLL) return fail(QW_EUNSUPPORTED, "lattice too large for one launch");
    long long blocks = (a.total_tiles + BLK1D_WARPS - 1) / BLK1D_WARPS;
    long long resident = (long long)s->sm_count * ctas_per_sm;
    if (s->max_ctas > 0 && resident > s->max_ctas) resident = s->max_ctas;
    if (blocks > resident) blocks = resident;
    kern<<<(unsigned)blocks, BLK1D_WARPS * 32, smem, s->stream>>>(a);
    QW_LAUNCH_CHECK(s, "step_blocked1d_kernel");
    return QW_OK;
}

template <typename R, int M, int KIND>
static int launch_blocked1d_t(qw_sim *s, const void *in, void *out, int k) {
    typedef typename Cx<R>::T V;
    const Geom &g = s->g;
    Blocked1dArgs<R> a;
    a.in = static_cast<const V *>(in);
    a.out = static_cast<V *>(out);
    a.n_sites = g.en; a.walk_stride = g.walk_stride; a.plane_stride = g.plane_stride;
    a.k = k; a.valid = 32 * M - 2 * k;
    a.tiles_per_walk = (g.en + a.valid - 1) / a.valid;
    a.total_tiles = a.tiles_per_walk * g.batch;
    a.boundary = g.boundary;
    for (int i = 0; i < 8; ++i) a.coin[i] = (R)s->h_coin[i];
    R sm = (R)1;
    for (int i = 0; i < M; ++i) sm = (R)(sm * a.coin[0]);    // s^M by repeated rounded products in the handle's precision
    a.scale_m = sm;
    if (g.boundary == QW_OPEN) return launch_blocked1d_k<R, M, KIND, true>(s, a);
    return launch_blocked1d_k<R, M, KIND, false>(s, a);
}

// Sites per lane: larger M = larger tiles (better valid fraction) but more registers and code.  The main launches use
// M = 16 (Hadamard) / 8 (general coin) and depths that are multiples of M; a remainder of 4 .. 15 steps is mopped up by
// one or two short launches with M = 8 / M = 4 tiles (one HBM round trip instead of 8 / 4 fused single steps).
int blocked1d_granule(const qw_sim *s) {
    return s->coin_kind == COIN_HADAMARD ? 16 : 8;
}

bool blocked1d_eligible(const qw_sim *s) {
    const Geom &g = s->g;
    return g.dim == 1 && s->coin_mode == QW_COIN_UNIFORM && !s->d_phases && !s->d_broken && !s->rbl &&
           g.en >= 32LL * blocked1d_granule(s);
}

// Tile computations per warp of one k-step launch (the halo kernel recomputes 2k of every 32*M sites).
double blocked1d_cost(const qw_sim *s, int k) {
    const int M = (s->coin_kind == COIN_HADAMARD && k % 16 == 0) ? 16 : (k % 8 == 0 ? 8 : 4);
    const long long valid = 32LL * M - 2LL * k;
    if (valid <= 0) return 1e300;
    const long long tiles = (s->g.en + valid - 1) / valid * s->g.batch;
    long long ctas = (long long)s->sm_count * (s->dtype == QW_C128 ? 2 : 4);
    if (s->max_ctas > 0 && ctas > s->max_ctas) ctas = s->max_ctas;
    const long long warps = ctas * BLK1D_WARPS;
    return (double)((tiles + warps - 1) / warps);
}

int blocked1d_max_k(const qw_sim *s) {
    // keep at least half of every tile valid: 2k <= 16*M
    return 8 * blocked1d_granule(s);
}

template <typename R>
static int launch_blocked1d_r(qw_sim *s, const void *in, void *out, int k) {
    const bool had = s->coin_kind == COIN_HADAMARD;
    const int M = (had && k % 16 == 0) ? 16 : (k % 8 == 0 ? 8 : 4);
    if (k <= 0 || k % M != 0 || 2 * k >= 32 * M) return fail(QW_EINVAL, "blocked step depth %d invalid for tile granule %d", k, M);
    if (had) {
        if (M == 16) return launch_blocked1d_t<R, 16, COIN_HADAMARD>(s, in, out, k);
        if (M == 8) return launch_blocked1d_t<R, 8, COIN_HADAMARD>(s, in, out, k);
        return launch_blocked1d_t<R, 4, COIN_HADAMARD>(s, in, out, k);
    }
    if (M == 8) return launch_blocked1d_t<R, 8, COIN_GENERAL>(s, in, out, k);
    return launch_blocked1d_t<R, 4, COIN_GENERAL>(s, in, out, k);
}

int launch_step_blocked1d(qw_sim *s, const void *in, void *out, int k) {
    return s->dtype == QW_C128 ? launch_blocked1d_r<double>(s, in, out, k) : launch_blocked1d_r<float>(s, in, out, k);
}

}  // namespace qw
