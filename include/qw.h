/* qw.h — C ABI of libqw: B200-native discrete-time coined quantum walk on Z^1 / Z^2.
 *
 * The library computes the repeated one-step evolution
 *
 *        psi(t+1) = U psi(t),      U = S (I (x) C)          (eq. 2; eq. 7)
 *
 * of Sawerwain & Gielerak, "GPGPU based simulations for one and two dimensional quantum walks"
 * (arXiv 1003.3779): a local unitary coin C_v acts on every site's coin space (PAPER.md:35-38
 * eq. 1), then the conditional shift S moves every coin component to its neighbour site
 * (eq. 3; eq. 8), and finally the per-vertex probability
 * distribution is formed by marginalising over the coin (Figs. 3-4).
 * Every step of that path runs in hand-written CUDA kernels for sm_100a; there is no CPU
 * fallback: every call returns QW_ECUDA when no device is usable.
 *
 * Conventions (DESIGN.md "Readings of the paper" lists each with its justification)
 *   site index     1D: x in [0, extents[0]);  2D: m * extents[1] + n  (n fastest)
 *   coin index     1D: 0 = R moves x -> x+1, 1 = L moves x -> x-1
 *                  2D: c = 2j + k for the paper's |j,k>; QW_NATURAL lattice      (eq. 8)
 *                        c0 -> (m, n+1)   c1 -> (m+1, n)   c2 -> (m-1, n)   c3 -> (m, n-1)
 *                      QW_DIAGONAL lattice (Fig. 1c): (m + (-1)^j, n + (-1)^k)
 *   one step       coin first, then shift
 *   QW_PERIODIC    site indices taken modulo the extents
 *   QW_OPEN        the links leaving the lattice are broken (RBL = 0 in PAPER.md:94-101,
 *                  eqs. 9-10): the component stays on its site with the opposite coin
 *                  (1D: 1-a; 2D: 3-c), no sign change.  U stays unitary.
 *   complex        interleaved (re, im); QW_C128 = 2 x double, QW_C64 = 2 x float; coin
 *                  matrices, phases and coin vectors use the dtype of the handle
 *   user layout    "AoS": [batch][site][coin] complex.  The device layout (one plane per coin
 *                  direction, PAPER-independent design choice) is private to the handle.
 *
 * Pointers: every data pointer (`const void *` / `void *` / `double *` / `uint8_t *`) may be a
 * host pointer (pageable or pinned) or a device pointer; the library classifies it with
 * cudaPointerGetAttributes.  Reading from / writing to host memory synchronises the handle's
 * stream before the call returns; with device pointers the call is asynchronous on that
 * stream.  `extents`, `site` and `qw_get_info`'s `out` are always host pointers.
 *
 * Ownership: the handle owns its device state (allocated by qw_create*, freed by qw_destroy).
 * Callers own every buffer they pass; host buffers may be reused when the call returns,
 * device buffers once the stream has passed the call.
 *
 * Errors: every call returns QW_OK (0) or a negative code, never throws or aborts; after an
 * error the handle is unchanged (except QW_ECUDA raised by an asynchronous failure).
 * qw_last_error() returns a thread-local message for the last non-zero return.
 * A handle must not be used from two host threads at the same time.  A handle belongs to the CUDA device that was
 * current when it was created; calls that touch its state return QW_EINVAL while another device is current.
 */
#ifndef QW_H_
#define QW_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qw_sim qw_sim;

enum { QW_OK = 0, QW_EINVAL = -1, QW_ENOMEM = -2, QW_ECUDA = -3, QW_ESTATE = -4, QW_EUNSUPPORTED = -5 };
enum { QW_C64 = 0, QW_C128 = 1 };
enum { QW_PERIODIC = 0, QW_OPEN = 1 };
enum { QW_NATURAL = 0, QW_DIAGONAL = 1 };
enum { QW_COIN_UNIFORM = 0, QW_COIN_PER_WALK = 1, QW_COIN_PER_SITE = 2 };

/* Step schedules (qw_set_schedule). */
enum {
    QW_SCHED_AUTO = 0,     /* library picks: resident if a walk fits one CTA, else blocked (1D) / tiled
                              (2D) / fused.  All schedules give bit-identical states except the blocked 1D
                              schedule with the Hadamard coin, whose scale is applied once per 16 steps
                              (<= 4 ulp per step from the others)                    */
    QW_SCHED_GENERIC = 1,  /* one launch per step, one thread per site, every feature (reference kernel) */
    QW_SCHED_FUSED = 2,    /* one launch per step, vectorised fused coin+shift (HBM-bound)              */
    QW_SCHED_BLOCKED = 3,  /* temporally blocked: k steps per HBM round trip (1D: register tiles per warp —
                              on a ring chained through the stream of L amplitudes, no halo recomputation;
                              2D: shared-memory tiles loaded by TMA)                                    */
    QW_SCHED_RESIDENT = 4, /* one CTA per walk, state on the SM for all n steps                         */
    QW_SCHED_TILED = 5     /* 2D temporally blocked with the state of k steps held in REGISTERS; honours the
                              light-cone window.  Natural lattice, any boundary: every warp streams down a strip
                              of columns with a k-level pipeline of rows in its registers (no halo along m, no
                              barriers; k even, <= 10 for complex64, <= 8 for complex128, <= 6 with random broken links), or — QW_OPT_TILED2D_KERNEL
                              — tiles held by persistent CTAs with TMA prefetch (k in {2, 4, 6, 8}).  Diagonal
                              lattice (tiles only): torus, or open lattice after qw_set_state_delta (the fused
                              kernel takes over when the cone reaches a wall)                                  */
};

/* qw_get_info keys */
enum {
    QW_INFO_LAUNCHES = 0,       /* kernels launched by this handle so far                                */
    QW_INFO_TIME = 1,           /* net number of steps applied since the last qw_set_state*              */
    QW_INFO_LAST_SCHEDULE = 2,  /* schedule the last qw_step actually used (QW_SCHED_*)                   */
    QW_INFO_LAST_K = 3,         /* temporal block depth of the last qw_step (1 if not blocked)           */
    QW_INFO_STATE_BYTES = 4,    /* bytes of one device state buffer (there are two)                      */
    QW_INFO_WINDOW = 5,         /* 1 if the light-cone window is active                                  */
    QW_INFO_SITES_TOUCHED = 6   /* site-steps the kernels were asked to produce so far: with the light-cone
                                   window only the sites / tiles / warps that were not skipped count; halo
                                   recomputation does not.  Without a window = batch * sites * steps          */
};

/* qw_set_option keys */
enum {
    QW_OPT_MAX_CTAS = 0,        /* cap on the grid of the persistent (blocked 1D) kernels; 0 = one grid
                                   that fills every SM (default).  For sharing a GPU and for tests that want
                                   long per-warp tile chains on small lattices; results do not depend on it */
    QW_OPT_BLOCKED1D_KERNEL = 1,/* which temporally blocked 1D kernel QW_SCHED_BLOCKED uses on a ring: 0 = the
                                   cheaper one (default), 1 = warp tiles with recomputed halos, 2 = chained
                                   tiles (no halo work; rings with a uniform coin, else falls back to 1).
                                   Both execute the same arithmetic per site: bit-identical results          */
    QW_OPT_TILED2D_KERNEL = 2   /* which register-resident 2D kernel QW_SCHED_TILED uses on the natural lattice:
                                   0 = the streaming kernel (default), 1 = CTA tiles with TMA prefetch,
                                   2 = the streaming kernel.  Bit-identical results                         */
};

/* Create a walk on a dim-dimensional lattice (dim = 1 or 2) with `extents[d] >= 1` sites per
 * axis.  coin_dim must equal 2*dim (degree of every vertex) else QW_EINVAL.
 * qw_create == qw_create_batch(1, ...).  A batch holds `batch` independent walks on identical
 * lattices (coin families may differ per walk and per vertex).
 * On success *out is a new handle on the current CUDA device, stream 0, no coin, no state. */
int qw_create(int dim, const int64_t *extents, int coin_dim, int dtype, int boundary, qw_sim **out);
int qw_create_batch(int64_t batch, int dim, const int64_t *extents, int coin_dim, int dtype,
                    int boundary, qw_sim **out);
int qw_destroy(qw_sim *s);

/* All later work of the handle is issued on `cuda_stream` (a cudaStream_t, e.g.
 * torch.cuda.current_stream().cuda_stream; NULL = default stream). */
int qw_set_stream(qw_sim *s, void *cuda_stream);

/* 2D only: QW_NATURAL (default, eq. 8) or QW_DIAGONAL (Fig. 1c, the
 * lattice of the paper's Tables 2-3). */
int qw_set_lattice(qw_sim *s, int lattice);

/* Coin family C = (C_v) (eq. 1).  `coin`: row-major coin_dim x coin_dim complex
 * matrices, rows = output component: 1 matrix (UNIFORM), batch matrices (PER_WALK) or
 * batch*sites matrices (PER_SITE, [walk][site]).  The library does not check unitarity. */
int qw_set_coin(qw_sim *s, int mode, const void *coin);

/* Optional unit-modulus multipliers [batch][site] applied on top of a UNIFORM / PER_WALK coin:
 * C_{w,x} = phases[w][x] * C_w (BASELINE.json:configs[4]).  NULL removes them. */
int qw_set_site_phases(qw_sim *s, const void *phases);

/* Optional static broken links: mask[batch][site][coin] bytes, non-zero =
 * the link that component `coin` of `site` would cross is broken; the component then stays on
 * the site with the opposite coin (eq. 10 with RBL = 0).  Both ends of a link must carry the
 * same bit (not checked).  NULL removes the mask. */
int qw_set_broken_links(qw_sim *s, const uint8_t *mask);

/* Random broken links redrawn at EVERY step ("random broken links (termed RBL) technique";
 * PAPER.md:92-102 eqs. 9-10): with enable != 0, step t (t = steps applied since the last qw_set_state*)
 * applies U(t) in which every link of the lattice is broken independently with probability p in [0, 1];
 * a broken link acts as in qw_set_broken_links.  The paper names no generator; the state of a link is
 * the pure function (reading R27)
 *     number  =  owner * dim + axis                      (dim = links a site owns: 1 in 1D, 2 in 2D)
 *     broken  <=>  Philox4x32-10(counter = (number/4 lo32, number/4 hi32, t lo32, walk lo32), key = seed)[number mod 4]
 *                  < floor(p * 2^32)
 * (one generator call serves four consecutive links with its four output words).
 * owner = site index of the end from which the link points in the positive direction (dm > 0, or
 * dm = 0 and dn > 0); axis = 0 for links along n (1D, natural) or along (+1,+1) (diagonal), 1 for links
 * along m or along (+1,-1).  Both ends of a link see the same value, so every U(t) is unitary, and
 * qw_step_inverse undoes the same sequence (QW_ESTATE if it would pass t = 0).  Links leaving a QW_OPEN
 * lattice stay broken; a static mask, if set, is OR-ed in.  enable = 0 switches the redraw off.
 * QW_EINVAL for p outside [0, 1]. */
int qw_set_random_broken_links(qw_sim *s, int enable, double p, uint64_t seed);

/* Set the state from AoS amplitudes [batch][site][coin]; resets the step counter.  The library
 * never normalises (eq. 4 is the caller's responsibility). */
int qw_set_state(qw_sim *s, const void *amps);

/* Every walk of the batch: zero everywhere, `coin_vec` (coin_dim complex) at `site` (dim indices).
 * Makes the light-cone window (eqs. 13-15, 17-18) available. */
int qw_set_state_delta(qw_sim *s, const int64_t *site, const void *coin_vec);

/* Copy the state out as AoS [batch][site][coin]. */
int qw_get_state(const qw_sim *s, void *amps);

/* n >= 0 applications of U (n = 0 is a no-op), asynchronous on the handle's stream.
 * QW_ESTATE before qw_set_coin or qw_set_state*; QW_EINVAL for n < 0. */
int qw_step(qw_sim *s, int64_t n);

/* n applications of U^dagger = (I (x) C^dagger) S^dagger (reversibility checks). */
int qw_step_inverse(qw_sim *s, int64_t n);

/* P[w][x] = sum_a |psi[w][x][a]|^2: [batch][site] double (C128) / float (C64). */
int qw_probabilities(const qw_sim *s, void *out);

/* Ensemble average over the batch: out[x] = (1 / batch) * sum_walks P_walk(x), `sites` reals of the handle's real type
 * (host or device), sites in row-major order.  This is the averaged distribution of the random-broken-links model
 * ("random broken links (termed RBL) technique", :221 "without and with broken links"): with
 * qw_set_random_broken_links every walk of a batch draws its own links, so a batch started from one initial state is
 * an ensemble of realisations.  Accumulated in double over the walks in order (deterministic).
 * QW_ESTATE without a state. */
int qw_probabilities_mean(const qw_sim *s, void *out);

/* Per walk, in double regardless of dtype: 1D {norm, mean, var};
 * 2D {norm, mean_m, mean_n, var_m, var_n, cov_mn}.  Coordinates x_d = index_d - floor(extent_d/2);
 * mean and (population) variance are divided by the computed norm (eq. 4 fixes norm = 1). */
int qw_moments(const qw_sim *s, double *out);

/* qw_moments for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): same kernels, same result layout, but the block partial sums live in a static device array of the library
 * (512 KiB, held by every GPU that loads the library until exit) instead of a lazily grown cudaMalloc buffer, and `out`
 * must be DEVICE memory (batch * 3 doubles in 1D, batch * 6 in 2D); the call performs no cudaMalloc / cudaFree and is
 * asynchronous on the handle's stream.  Limit: batch <= 8192 walks, else QW_EUNSUPPORTED; QW_EINVAL for a host `out`.
 * The blocks per walk are capped by the array, so the summation order — and the last bits of the result — can differ
 * from qw_moments (same tolerance against the definition).  All calls on a device SHARE the array: calls in one stream are
 * safe back to back (each call rewrites every entry it reads), calls that overlap on the GPU (other streams, other
 * handles) race. */
int qw_moments_static(const qw_sim *s, double *out);

/* Force a schedule (QW_SCHED_*); k = temporal block depth for QW_SCHED_BLOCKED / QW_SCHED_TILED
 * (0 = library default; QW_SCHED_TILED accepts the even depths listed at QW_SCHED_TILED, else QW_EINVAL).
 * QW_EUNSUPPORTED if the handle's configuration has no such kernel. */
int qw_set_schedule(qw_sim *s, int schedule, int k);

/* Enable (1, default) / disable (0) the light-cone window: after qw_set_state_delta only sites
 * within t+1 of the start are updated at step t.  Exact: skipped sites are 0. */
int qw_set_window(qw_sim *s, int enable);

/* Tuning knobs that never change results (QW_OPT_*).  QW_EINVAL for an unknown key or a bad value. */
int qw_set_option(qw_sim *s, int key, int64_t value);

int qw_get_info(const qw_sim *s, int what, int64_t *out);

/* Diagnostic for the roofline of the schedules that are not HBM-bound (temporally blocked, resident): the measured
 * plain-ALU throughput of the current device for the instructions the coin arithmetic is made of (PAPER.md:37-38
 * eq. 1 evaluated as additions and fused multiply-adds, csrc/qw_coin.cuh).  dtype QW_C128: FP64 (DADD / DFMA);
 * QW_C64: packed FP32x2 (FADD2 / FFMA2).  op: QW_PEAK_ADD or QW_PEAK_FMA.  Runs a register-only kernel on every
 * SM of the current device (default stream, synchronous, a few milliseconds) and stores thread-level operations per
 * second (an FMA counts as ONE operation, a packed instruction as two) in *ops_per_second (host pointer).
 * No handle, no walk arithmetic. */
enum { QW_PEAK_ADD = 0, QW_PEAK_FMA = 1 };
int qw_measure_alu_peak(int dtype, int op, double *ops_per_second);

/* Block the host until the handle's stream is idle; reports asynchronous CUDA errors. */
int qw_synchronize(const qw_sim *s);

const char *qw_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* QW_H_ */
