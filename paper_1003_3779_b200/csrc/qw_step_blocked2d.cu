// qw_step_blocked2d.cu — temporally blocked 2D step: k applications of U = S (C (x) I)
// (eq. 7 with the shift of PAPER.md:88 eq. 8) per HBM round trip, uniform coin,
// natural lattice.
//
// A CTA stages a tile of HM x HN sites of all four coin planes (valid interior (HM-2k) x (HN-2k) plus a
// k-site halo: after k steps the unknown outside has travelled exactly k sites inwards
// eq. 18) in shared memory with ONE TMA box load per plane (cp.async.bulk.tensor.3d + mbarrier), then
// advances k steps in shared memory and stores the valid interior.
//
// In-place co-moving update: plane c is kept in the frame that moves with its own shift, i.e. after
// s steps the amplitude psi_c(x) is stored at tile location x - s*d_c.  One step for site x then reads
// the four locations x - s*d_c, applies the coin (eq. 1) and writes the results back to THE SAME
// locations, which in the next frame are exactly the shifted amplitudes (eq. 8).  No ping-pong copy of
// the tile, no data movement for the shift; one __syncthreads per step.  Rows [s, HM-s) are processed at
// step s, so every location touched stays inside the tile.
//
// Halos: every 2D state buffer carries a ghost ring of QW_GHOST_2D cells (qw_internal.cuh).  On a
// periodic lattice it is refreshed from the opposite edges before each blocked launch, so every tile
// is one plain in-bounds box; beyond the allocation TMA zero-fills.  On an open lattice (reflecting
// walls = broken outward links) sites outside the lattice are never stored and the
// wall sites write the reflected component into the opposite plane's next-frame location.
// The halo is k sites (k+1 for complex64 with odd k: the TMA box origin must be 16-byte aligned).
#include <cuda.h>

#include "qw_coin.cuh"

namespace qw {

constexpr int B2D_THREADS = 512;
constexpr int B2D_WARPS = B2D_THREADS / 32;

template <typename R>
struct Blocked2dArgs {
    typename Cx<R>::T *out;       // site (0,0) of walk 0, plane 0 of the output buffer
    long long em, en, pitch, walk_stride, plane_stride;
    int batch, k, halo, ghost, tiles_n, tiles_m;   // halo >= k sites around the valid interior
    R coin[32];
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}

template <typename R, int KIND, bool OPEN, int HM, int HN>
__global__ void __launch_bounds__(B2D_THREADS)
step_blocked2d_kernel(const __grid_constant__ CUtensorMap tmap, const Blocked2dArgs<R> a) {
    typedef typename Cx<R>::T V;
    static_assert(HN % 32 == 0, "tile width must be a multiple of the warp size");
    constexpr int CPR = HN / 32;                 // 32-site chunks per tile row
    constexpr int PLANE = HM * HN;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    V *A = reinterpret_cast<V *>(smem_raw);      // A[c * PLANE + row * HN + col]
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + (size_t)4 * PLANE * sizeof(V));

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int k = a.k, halo = a.halo;
    const int TM = HM - 2 * halo, TN = HN - 2 * halo;
    const int w = blockIdx.z;
    const long long m0 = (long long)blockIdx.y * TM - halo;  // lattice coordinates of tile location (0,0)
    const long long n0 = (long long)blockIdx.x * TN - halo;

    if (tid == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(bar, (uint32_t)(4 * PLANE * sizeof(V)));
        const int c0 = (int)(n0 + a.ghost) * (int)(sizeof(V) / 8);   // inner dimension counts 8-byte words
        const int c1 = (int)(m0 + a.ghost);
#pragma unroll
        for (int c = 0; c < 4; ++c) tma_load_3d(A + c * PLANE, &tmap, c0, c1, c * a.batch + w, bar);
    }
    const R *C = a.coin;                         // kernel parameter = constant bank operands
    mbar_wait(bar, 0);

    bool wall_tile = false;
    if (OPEN) wall_tile = (m0 < 0) || (n0 < 0) || (m0 + HM > a.em) || (n0 + HN > a.en);

    for (int s = 0; s < k; ++s) {
        const int ntasks = (HM - 2 * s) * CPR;
        const int o0 = -s, o1 = -s * HN, o2 = s * HN, o3 = s;     // x - s*d_c for c = 0..3
        for (int task = wid; task < ntasks; task += B2D_WARPS) {
            const int row = s + task / CPR;
            const int col = (task % CPR) * 32 + lane;
            const int idx = row * HN + col;
            if (OPEN && wall_tile) {
                const long long gm = m0 + row, gn = n0 + col;
                if (gm < 0 || gm >= a.em || gn < 0 || gn >= a.en) continue;     // outside the lattice: never stored
                cplx<R> v[4];
                v[0] = cx_load<R>(A + 0 * PLANE + idx + o0);
                v[1] = cx_load<R>(A + 1 * PLANE + idx + o1);
                v[2] = cx_load<R>(A + 2 * PLANE + idx + o2);
                v[3] = cx_load<R>(A + 3 * PLANE + idx + o3);
                apply_coin<R, 4, KIND>(C, v);
                // c0 -> n+1, c1 -> m+1, c2 -> m-1, c3 -> n-1; a broken (outward) link keeps the component
                // on the site with the opposite coin: next-frame location of plane 3-c is x + (s+1) d_c
                const bool out0 = gn + 1 >= a.en, out1 = gm + 1 >= a.em, out2 = gm - 1 < 0, out3 = gn - 1 < 0;
                const int r0 = idx + (s + 1), r1 = idx + (s + 1) * HN, r2 = idx - (s + 1) * HN, r3 = idx - (s + 1);
                if (!out0) cx_store<R>(A + 0 * PLANE + idx + o0, v[0]);
                else if (r0 < PLANE) cx_store<R>(A + 3 * PLANE + r0, v[0]);
                if (!out1) cx_store<R>(A + 1 * PLANE + idx + o1, v[1]);
                else if (r1 < PLANE) cx_store<R>(A + 2 * PLANE + r1, v[1]);
                if (!out2) cx_store<R>(A + 2 * PLANE + idx + o2, v[2]);
                else if (r2 >= 0) cx_store<R>(A + 1 * PLANE + r2, v[2]);
                if (!out3) cx_store<R>(A + 3 * PLANE + idx + o3, v[3]);
                else if (r3 >= 0) cx_store<R>(A + 0 * PLANE + r3, v[3]);
            } else {
                cplx<R> v[4];
                v[0] = cx_load<R>(A + 0 * PLANE + idx + o0);
                v[1] = cx_load<R>(A + 1 * PLANE + idx + o1);
                v[2] = cx_load<R>(A + 2 * PLANE + idx + o2);
                v[3] = cx_load<R>(A + 3 * PLANE + idx + o3);
                apply_coin<R, 4, KIND>(C, v);
                cx_store<R>(A + 0 * PLANE + idx + o0, v[0]);
                cx_store<R>(A + 1 * PLANE + idx + o1, v[1]);
                cx_store<R>(A + 2 * PLANE + idx + o2, v[2]);
                cx_store<R>(A + 3 * PLANE + idx + o3, v[3]);
            }
        }
        __syncthreads();
    }

    // store the valid interior: psi_c(x) sits at location x - k*d_c
    const int q0 = -k, q1 = -k * HN, q2 = k * HN, q3 = k;
    V *outw = a.out + (long long)w * a.walk_stride;
    const int cps = (TN + 31) / 32;
    for (int task = wid; task < TM * cps; task += B2D_WARPS) {
        const int row = halo + task / cps;
        const int col = halo + (task % cps) * 32 + lane;
        const long long gm = m0 + row, gn = n0 + col;
        if (col < HN - halo && gm < a.em && gn < a.en) {
            const int idx = row * HN + col;
            const long long g = gm * a.pitch + gn;
            outw[0 * a.plane_stride + g] = A[0 * PLANE + idx + q0];
            outw[1 * a.plane_stride + g] = A[1 * PLANE + idx + q1];
            outw[2 * a.plane_stride + g] = A[2 * PLANE + idx + q2];
            outw[3 * a.plane_stride + g] = A[3 * PLANE + idx + q3];
        }
    }
}

// Periodic lattices: fill the ghost ring of every plane / walk from the opposite edges.
template <typename V>
__global__ void ghost_refresh_kernel(V *base /* allocation start of plane 0 */, long long em, long long en, long long pitch,
                                     long long walk_stride, int ghost, long long nwalkplanes) {
    // frame cells in padded coordinates (pm, pn) in [0, em+2g) x [0, en+2g) that are not interior
    const long long PM = em + 2 * ghost, PN = en + 2 * ghost;
    const long long top = (long long)ghost * PN;                 // rows above
    const long long side = em * 2LL * ghost;                     // left + right strips of the interior rows
    const long long per = 2 * top + side;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= per) return;
    long long pm, pn;
    if (i < top) { pm = i / PN; pn = i - pm * PN; }
    else if (i < 2 * top) { const long long j = i - top; pm = ghost + em + j / PN; pn = j - (j / PN) * PN; }
    else { const long long j = i - 2 * top; pm = ghost + j / (2 * ghost); const long long q = j - (j / (2 * ghost)) * (2 * ghost);
           pn = q < ghost ? q : en + q; }
    long long sm = (pm - ghost) % em; if (sm < 0) sm += em;
    long long sn = (pn - ghost) % en; if (sn < 0) sn += en;
    for (long long wp = blockIdx.y; wp < nwalkplanes; wp += gridDim.y) {
        V *p = base + wp * walk_stride;
        p[pm * pitch + pn] = p[(sm + ghost) * pitch + (sn + ghost)];
    }
    (void)PM;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// Tile geometry per dtype: two CTAs per SM (<= ~100 KB each) so that one tile's TMA load / store
// overlaps the other's compute.
template <typename R> struct B2dTile;
template <> struct B2dTile<float>  { static constexpr int HM = 48, HN = 64; };   // 48*64*32 B = 96 KiB
template <> struct B2dTile<double> { static constexpr int HM = 24, HN = 64; };   // 24*64*64 B = 96 KiB

static int tile_hm(const qw_sim *s) { return s->dtype == QW_C128 ? B2dTile<double>::HM : B2dTile<float>::HM; }
static int tile_hn(const qw_sim *s) { return s->dtype == QW_C128 ? B2dTile<double>::HN : B2dTile<float>::HN; }

static int build_tmaps(qw_sim *s) {
    if (s->tmap_ready) return QW_OK;
    EncodeTiledFn enc = encode_fn();
    if (!enc) return fail(QW_ECUDA, "cuTensorMapEncodeTiled is not available from this driver");
    const Geom &g = s->g;
    const cuuint64_t words = s->esize / 8;                     // 8-byte words per complex
    const cuuint64_t dims[3] = {(cuuint64_t)g.pitch * words, (cuuint64_t)(g.em + 2 * g.ghost), (cuuint64_t)(4 * g.batch)};
    const cuuint64_t strides[2] = {(cuuint64_t)g.pitch * s->esize, (cuuint64_t)g.walk_stride * s->esize};
    const cuuint32_t box[3] = {(cuuint32_t)(tile_hn(s) * words), (cuuint32_t)tile_hm(s), 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    for (int i = 0; i < 2; ++i) {
        CUresult r = enc(reinterpret_cast<CUtensorMap *>(s->tmap[i]), CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, s->buf[i], dims, strides, box,
                         estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(QW_ECUDA, "cuTensorMapEncodeTiled failed with code %d", (int)r);
    }
    s->tmap_ready = true;
    return QW_OK;
}

bool blocked2d_eligible(const qw_sim *s) {
    const Geom &g = s->g;
    return g.dim == 2 && g.lattice == QW_NATURAL && s->coin_mode == QW_COIN_UNIFORM && !s->d_phases && !s->d_broken && !s->rbl &&
           g.em >= 2 * QW_GHOST_2D && g.en >= 2 * QW_GHOST_2D && g.batch <= 16383 && g.walk_stride * 4 * g.batch < (1LL << 40);
}

int blocked2d_max_k(const qw_sim *s) {
    const int lim = (tile_hm(s) - 2) / 2;                      // at least two valid rows
    return lim < QW_GHOST_2D ? lim : QW_GHOST_2D;
}

template <typename R, int KIND>
static int launch_blocked2d_t(qw_sim *s, int in_buf, int out_buf, int k) {
    typedef typename Cx<R>::T V;
    constexpr int HM = B2dTile<R>::HM, HN = B2dTile<R>::HN;
    const Geom &g = s->g;
    Blocked2dArgs<R> a;
    a.out = static_cast<V *>(state_ptr(s, out_buf));
    a.em = g.em; a.en = g.en; a.pitch = g.pitch; a.walk_stride = g.walk_stride; a.plane_stride = g.plane_stride;
    a.batch = (int)g.batch; a.k = k; a.ghost = g.ghost;
    // TMA needs a 16-byte aligned box origin: with 8-byte complex64 elements the halo must be even
    a.halo = (sizeof(V) == 8 && (k & 1)) ? k + 1 : k;
    const int TM = HM - 2 * a.halo, TN = HN - 2 * a.halo;
    a.tiles_m = (int)((g.em + TM - 1) / TM); a.tiles_n = (int)((g.en + TN - 1) / TN);
    for (int i = 0; i < 32; ++i) a.coin[i] = (R)s->h_coin[i];
    const size_t smem = (size_t)4 * HM * HN * sizeof(V) + 16;
    dim3 grid((unsigned)a.tiles_n, (unsigned)a.tiles_m, (unsigned)g.batch);
    if (a.tiles_m > 65535) return fail(QW_EUNSUPPORTED, "lattice too tall for the blocked 2D launch");
    const CUtensorMap &tm = *reinterpret_cast<const CUtensorMap *>(s->tmap[in_buf]);
    auto go = [&](auto kernel) -> int {
        QW_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kernel<<<grid, B2D_THREADS, smem, s->stream>>>(tm, a);
        return QW_OK;
    };
    int rc = g.boundary == QW_OPEN ? go(step_blocked2d_kernel<R, KIND, true, HM, HN>)
                                   : go(step_blocked2d_kernel<R, KIND, false, HM, HN>);
    if (rc) return rc;
    QW_LAUNCH_CHECK(s, "step_blocked2d_kernel");
    return QW_OK;
}

int launch_ghost_refresh(qw_sim *s, int buf) {
    const Geom &g = s->g;
    const long long per = 2LL * g.ghost * (g.en + 2 * g.ghost) + g.em * 2LL * g.ghost;
    const long long nwp = 4 * g.batch;
    dim3 grid((unsigned)((per + 255) / 256), (unsigned)(nwp < 64 ? nwp : 64));
    if (s->dtype == QW_C128)
        ghost_refresh_kernel<double2><<<grid, 256, 0, s->stream>>>(static_cast<double2 *>(s->buf[buf]), g.em, g.en, g.pitch,
                                                                   g.walk_stride, g.ghost, nwp);
    else
        ghost_refresh_kernel<float2><<<grid, 256, 0, s->stream>>>(static_cast<float2 *>(s->buf[buf]), g.em, g.en, g.pitch,
                                                                  g.walk_stride, g.ghost, nwp);
    QW_LAUNCH_CHECK(s, "ghost_refresh_kernel");
    return QW_OK;
}

// Natural lattice: as the shared-memory blocked kernel.  Diagonal lattice (no wall code): a torus, or an open lattice
// with a known light cone — then tiled2d_diag_open_ok() must hold for every launch.
bool tiled2d_eligible(const qw_sim *s) {
    if (blocked2d_eligible(s)) return true;
    const Geom &g = s->g;
    const bool base = g.dim == 2 && g.lattice == QW_DIAGONAL && s->coin_mode == QW_COIN_UNIFORM && !s->d_phases && !s->d_broken &&
                      !s->rbl && g.em >= 2 * QW_GHOST_2D && g.en >= 2 * QW_GHOST_2D && g.batch <= 16383 &&
                      g.walk_stride * 4 * g.batch < (1LL << 40);
    return base && (g.boundary == QW_PERIODIC || (s->window_enabled && s->window_valid));
}

// Open diagonal lattice: can k more steps be taken without any amplitude touching a wall?  The support after j steps
// lies within Chebyshev distance radius + j of the start; a reflection at step j needs a wall site inside it.
bool tiled2d_diag_open_ok(const qw_sim *s, int k) {
    const Geom &g = s->g;
    if (g.lattice != QW_DIAGONAL || g.boundary != QW_OPEN) return true;
    if (!(s->window_enabled && s->window_valid)) return false;
    long long d = s->centre[0];
    if (g.em - 1 - s->centre[0] < d) d = g.em - 1 - s->centre[0];
    if (s->centre[1] < d) d = s->centre[1];
    if (g.en - 1 - s->centre[1] < d) d = g.en - 1 - s->centre[1];
    return s->radius + k <= d;
}

// Register-tiled schedule: refresh the periodic halos, then dispatch on the dtype.
int launch_step_tiled2d(qw_sim *s, int in_buf, int out_buf, int k, const Box &box) {
    if (s->g.boundary == QW_PERIODIC) {
        int rc = launch_ghost_refresh(s, in_buf);
        if (rc) return rc;
    }
    return s->dtype == QW_C128 ? launch_tiled2d_f64(s, in_buf, out_buf, k, box) : launch_tiled2d_f32(s, in_buf, out_buf, k, box);
}

// Streaming schedule (qw_step_stream2d.cuh): natural lattice, uniform coin; same ghost ring as the tiles.
// Random broken links redrawn every step are drawn inside the kernel when the rows have even length (two sites of a
// lane share one generator call); depth <= 6 then.
bool stream2d_eligible(const qw_sim *s) {
    const Geom &g = s->g;
    return g.dim == 2 && g.lattice == QW_NATURAL && s->coin_mode == QW_COIN_UNIFORM && !s->d_phases && !s->d_broken &&
           (!s->rbl || g.en % 2 == 0) && g.em >= 2 * QW_GHOST_2D && g.en >= 2 * QW_GHOST_2D && g.batch <= 16383 &&
           g.walk_stride * 4 * g.batch < (1LL << 40);
}
int stream2d_max_k(const qw_sim *s) { return s->rbl ? 6 : (s->dtype == QW_C128 ? 8 : 10); }

// On a torus the units at the seams wrap their input rows and columns themselves when the rows have even length (a lane's
// two-column segment then never straddles the seam and stays 16-byte aligned); otherwise the halos come from the refreshed
// ghost ring.
bool stream2d_wraps(const qw_sim *s) { return s->g.boundary == QW_PERIODIC && s->g.en % 2 == 0; }

int launch_step_stream2d(qw_sim *s, int in_buf, int out_buf, int k, const Box &box) {
    if (s->g.boundary == QW_PERIODIC && !stream2d_wraps(s)) {
        int rc = launch_ghost_refresh(s, in_buf);
        if (rc) return rc;
    }
    if (s->rbl) return s->dtype == QW_C128 ? launch_stream2d_rbl_f64(s, in_buf, out_buf, k, box) : launch_stream2d_rbl_f32(s, in_buf, out_buf, k, box);
    return s->dtype == QW_C128 ? launch_stream2d_f64(s, in_buf, out_buf, k, box) : launch_stream2d_f32(s, in_buf, out_buf, k, box);
}

int launch_step_blocked2d(qw_sim *s, int in_buf, int out_buf, int k) {
    const Geom &g = s->g;
    if (k < 1 || k > blocked2d_max_k(s)) return fail(QW_EINVAL, "blocked 2D step depth %d outside [1, %d]", k, blocked2d_max_k(s));
    int rc = build_tmaps(s);
    if (rc) return rc;
    if (g.boundary == QW_PERIODIC) {
        rc = launch_ghost_refresh(s, in_buf);
        if (rc) return rc;
    }
#define QW_B2D(R)                                                                             \
    switch (s->coin_kind) {                                                                   \
        case COIN_GROVER4: return launch_blocked2d_t<R, COIN_GROVER4>(s, in_buf, out_buf, k); \
        case COIN_HXH4:    return launch_blocked2d_t<R, COIN_HXH4>(s, in_buf, out_buf, k);    \
        case COIN_DFT4:    return launch_blocked2d_t<R, COIN_DFT4>(s, in_buf, out_buf, k);    \
        default:           return launch_blocked2d_t<R, COIN_GENERAL>(s, in_buf, out_buf, k); \
    }
    if (s->dtype == QW_C128) { QW_B2D(double) }
    QW_B2D(float)
#undef QW_B2D
}

}  // namespace qw
