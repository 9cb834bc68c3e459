// qw_internal.cuh — private declarations shared by the translation units of libqw.
// Nothing here is part of the C ABI (include/qw.h) and nothing is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/qw.h"

namespace qw {

// ---------------------------------------------------------------------------------------------
// Device layout: structure of arrays, one contiguous complex
// plane per coin direction:  plane[c][walk][m][n_pitch].  Two such buffers (ping-pong).
// ---------------------------------------------------------------------------------------------
struct Geom {
    int dim;          // 1 or 2
    int cdim;         // 2 * dim
    int boundary;     // QW_PERIODIC / QW_OPEN
    int lattice;      // QW_NATURAL / QW_DIAGONAL
    long long batch;
    long long em, en;        // 1D: em = 1, en = extent
    long long sites;         // em * en
    long long pitch;         // complex elements per allocated row (>= en + 2*ghost, padded)
    long long walk_stride;   // (em + 2*ghost) * pitch
    long long plane_stride;  // batch * walk_stride
    int ghost;               // 2D: ghost ring of this many cells around every walk (0 in 1D); the
                             // temporally blocked 2D kernel reads its halos from it (periodic: refreshed
                             // from the opposite edge before every blocked launch; open: don't-care)
    long long origin;        // element offset of site (0,0) of walk 0 inside a plane: ghost*pitch + ghost
};

enum CoinKind {
    COIN_GENERAL = 0,   // full complex mat-vec
    COIN_HADAMARD = 1,  // 1D: s*[[1,1],[1,-1]], s real
    COIN_GROVER4 = 2,   // 2D: g*J - I-like: off-diagonal all equal real g, diagonal g-1... see qw_coin.cuh
    COIN_HXH4 = 3,      // 2D: h*[[1,1,1,1],[1,-1,1,-1],[1,1,-1,-1],[1,-1,-1,1]], h real
    COIN_DFT4 = 4       // 2D: h*i^(ab), h real
};

template <typename R> struct Cx;
template <> struct Cx<double> { typedef double2 T; };
template <> struct Cx<float>  { typedef float2 T; };

// Source-site box updated by one step (light-cone window).  Inclusive bounds.
struct Box { long long m_lo, m_hi, n_lo, n_hi; };

}  // namespace qw

// The opaque handle of include/qw.h.
struct qw_sim {
    qw::Geom g;
    int dtype;               // QW_C64 / QW_C128
    size_t esize;            // bytes per complex amplitude
    int device;
    int sm_count;
    cudaStream_t stream;

    void *buf[2];            // ping-pong state buffers, each cdim * plane_stride complex
    int cur;                 // buf[cur] holds psi(t)
    size_t state_bytes;

    // coin family
    bool has_coin;
    int coin_mode;
    int coin_kind;           // qw::CoinKind, classified from the uniform matrix
    double h_coin[32];       // uniform coin, complex interleaved, promoted to double
    void *d_coin;            // PER_WALK / PER_SITE matrices on the device (handle dtype)
    void *d_phases;          // optional [batch][site] complex multipliers
    uint8_t *d_broken;       // optional [batch][site][coin] link mask
    bool rbl;                // random broken links redrawn every step (qw_set_random_broken_links)
    uint64_t rbl_seed;
    uint64_t rbl_thr;        // floor(p * 2^32)

    // state bookkeeping
    bool has_state;
    long long t;             // net steps since set_state
    bool window_enabled;     // user switch
    bool window_valid;       // both buffers are zero outside the box below
    long long centre[2];
    long long radius;        // support of psi(t) is within `radius` of `centre` (Chebyshev)

    // schedule
    int max_ctas;            // QW_OPT_MAX_CTAS: cap on the grid of the persistent kernels (0 = all SMs)
    int blocked1d_kernel;    // QW_OPT_BLOCKED1D_KERNEL: 0 = cheaper of the two, 1 = halo tiles, 2 = chained tiles (rings)
    int tiled2d_kernel;      // QW_OPT_TILED2D_KERNEL: 0 = streaming kernel where it applies, 1 = register tiles, 2 = streaming
    int sched, sched_k;
    int last_sched, last_k;
    long long launches;
    double touched;          // site-steps the kernels were asked to produce so far (QW_INFO_SITES_TOUCHED): the sites
                             // inside the light-cone window / the tiles and warps that were not skipped; halo
                             // recomputation is not counted

    // TMA descriptors of the two state buffers (qw_step_blocked2d.cu), built lazily
    alignas(64) unsigned char tmap[2][128];
    bool tmap_ready;
    alignas(64) unsigned char tmap_t[2][128];   // ... of the register-tiled kernel (qw_step_tiled2d.cuh)
    bool tmap_t_ready;

    // host <-> device streaming of the state (qw_set_state / qw_get_state with host buffers): two staging buffers of
    // QW_STAGE_BYTES on the device, a private copy stream and events, so the PCIe copy of chunk i+1 overlaps the layout
    // kernel of chunk i and no state-sized scratch is needed
    void *stage[2];
    cudaStream_t copy_stream;
    cudaEvent_t ev_copy[2], ev_kernel[2];
    bool stage_ready;

    // scratch
    void *scratch;           // staging for outputs to host buffers (probabilities, moments)
    size_t scratch_bytes;
    double *partials;        // moment partial sums
    size_t partials_count;
};

namespace qw {

// pointer to site (0,0) of walk 0, plane 0 of state buffer i
inline void *state_ptr(const qw_sim *s, int i) {
    return static_cast<char *>(s->buf[i]) + (size_t)s->g.origin * s->esize;
}

// error reporting (qw_api.cu)
int fail(int code, const char *fmt, ...);
void clear_error();

#define QW_CUDA(call)                                                                         \
    do {                                                                                      \
        cudaError_t qw_e_ = (call);                                                           \
        if (qw_e_ != cudaSuccess)                                                             \
            return ::qw::fail(QW_ECUDA, "%s failed: %s", #call, cudaGetErrorString(qw_e_));   \
    } while (0)

#define QW_LAUNCH_CHECK(s, name)                                                              \
    do {                                                                                      \
        cudaError_t qw_e_ = cudaGetLastError();                                               \
        if (qw_e_ != cudaSuccess)                                                             \
            return ::qw::fail(QW_ECUDA, "launch of %s failed: %s", name,                      \
                              cudaGetErrorString(qw_e_));                                     \
        (s)->launches++;                                                                      \
    } while (0)

// ---- kernels' host-side launchers (one per translation unit) -------------------------------
// qw_layout.cu
int launch_aos_to_soa(qw_sim *s, const void *aos_dev, void *soa, long long first = 0, long long count = -1);
int launch_soa_to_aos(qw_sim *s, const void *soa, void *aos_dev, long long first = 0, long long count = -1);
int launch_delta(qw_sim *s, const long long *site, const double *coin_vec);

// qw_step.cu : one launch per step, scatter form.  fast = uniform coin, no phases, no links, natural.
int launch_step(qw_sim *s, const void *in, void *out, const Box &box, bool allow_fast);
int launch_step_inverse(qw_sim *s, const void *in, void *out);

// qw_step_blocked1d.cu : k steps per launch, warp-private register tiles (uniform coin, 1D)
bool blocked1d_eligible(const qw_sim *s);
int blocked1d_granule(const qw_sim *s);
int blocked1d_max_k(const qw_sim *s);
int launch_step_blocked1d(qw_sim *s, const void *in, void *out, int k);

// qw_step_chain1d.cu : k steps per launch on a ring, tiles chained through the stream of L amplitudes (no halo work)
bool chain1d_eligible(const qw_sim *s, int k);
int chain1d_granule(const qw_sim *s);
int chain1d_max_k(const qw_sim *s);
double chain1d_cost(qw_sim *s, int k);               // tile computations per warp of one launch
int launch_step_chain1d(qw_sim *s, const void *in, void *out, int k);
double blocked1d_cost(const qw_sim *s, int k);       // same for the halo kernel

// qw_step_resident1d.cu : one CTA per walk, all n steps on the SM (1D walks of <= 4096 sites)
bool resident1d_eligible(const qw_sim *s);
int launch_step_resident1d(qw_sim *s, const void *in, void *out, long long n);

// qw_step_blocked2d.cu : k steps per launch, shared-memory tiles loaded by TMA (uniform coin, 2D natural)
constexpr int QW_GHOST_2D = 16;
bool blocked2d_eligible(const qw_sim *s);
int blocked2d_max_k(const qw_sim *s);
int launch_step_blocked2d(qw_sim *s, int in_buf, int out_buf, int k);
int launch_ghost_refresh(qw_sim *s, int buf);     // periodic lattices: ghost ring := opposite edges

// qw_step_tiled2d_*.cu : k in {2,4,6,8} steps per launch, persistent CTAs, tiles in REGISTERS, TMA prefetch
// (uniform coin, 2D natural).  `box` = sites that can be non-zero after the launch (whole lattice if no window).
bool tiled2d_eligible(const qw_sim *s);
bool tiled2d_diag_open_ok(const qw_sim *s, int k);   // open diagonal lattice: k more steps cannot touch a wall
int launch_step_tiled2d(qw_sim *s, int in_buf, int out_buf, int k, const Box &box);
int launch_tiled2d_f32(qw_sim *s, int in_buf, int out_buf, int k, const Box &box);
int launch_tiled2d_f64(qw_sim *s, int in_buf, int out_buf, int k, const Box &box);

// qw_step_stream2d_*.cu : k in {2,..,12} (even) steps per launch, every warp streams down a strip of columns with a
// K-level pipeline of rows in REGISTERS (uniform coin, 2D natural lattice); the 2D AUTO schedule where it applies.
bool stream2d_eligible(const qw_sim *s);
int stream2d_max_k(const qw_sim *s);
bool stream2d_wraps(const qw_sim *s);   // torus: the kernel wraps its input addresses itself (no ghost-ring refresh before the launch)
int launch_step_stream2d(qw_sim *s, int in_buf, int out_buf, int k, const Box &box);
int launch_stream2d_f32(qw_sim *s, int in_buf, int out_buf, int k, const Box &box);
int launch_stream2d_f64(qw_sim *s, int in_buf, int out_buf, int k, const Box &box);
int launch_stream2d_rbl_f32(qw_sim *s, int in_buf, int out_buf, int k, const Box &box);   // random broken links drawn in the kernel
int launch_stream2d_rbl_f64(qw_sim *s, int in_buf, int out_buf, int k, const Box &box);

// qw_reduce.cu
int launch_probabilities(qw_sim *s, const void *state, void *out_dev);
int launch_probabilities_mean(qw_sim *s, const void *state, void *out_dev);   // [sites], mean over the batch
int launch_moments(qw_sim *s, const void *state, double *out_dev);
int launch_moments_static(qw_sim *s, const void *state, double *out_dev);   // partials in a static device array: no allocation

}  // namespace qw
