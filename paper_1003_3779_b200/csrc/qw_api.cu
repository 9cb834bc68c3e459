// qw_api.cu — the C ABI of include/qw.h: argument checking, device state ownership, host/device
// pointer handling and the schedule dispatcher.  All arithmetic of the walk lives in the kernels
// (qw_step*.cu, qw_reduce.cu); there is no CPU implementation of any step in this library.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "qw_internal.cuh"

namespace qw {

static thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}
void clear_error() { g_err[0] = 0; }

// true if p is device-accessible memory owned by the CUDA allocator (device or managed)
static bool is_device_ptr(const void *p) {
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

static int ensure_scratch(qw_sim *s, size_t bytes) {
    if (bytes <= s->scratch_bytes) return QW_OK;
    if (s->scratch) { cudaStreamSynchronize(s->stream); cudaFree(s->scratch); s->scratch = nullptr; s->scratch_bytes = 0; }
    cudaError_t e = cudaMalloc(&s->scratch, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(QW_ENOMEM, "cannot allocate %zu bytes of staging memory", bytes); }
    s->scratch_bytes = bytes;
    return QW_OK;
}

constexpr size_t QW_STAGE_BYTES = 64u << 20;

static int ensure_stage(qw_sim *s) {
    if (s->stage_ready) return QW_OK;
    for (int i = 0; i < 2; ++i) {
        if (cudaMalloc(&s->stage[i], QW_STAGE_BYTES) != cudaSuccess) {
            cudaGetLastError();
            if (i == 1) { cudaFree(s->stage[0]); s->stage[0] = nullptr; }
            return fail(QW_ENOMEM, "cannot allocate the %zu-byte staging buffers", QW_STAGE_BYTES);
        }
    }
    QW_CUDA(cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
        QW_CUDA(cudaEventCreateWithFlags(&s->ev_copy[i], cudaEventDisableTiming));
        QW_CUDA(cudaEventCreateWithFlags(&s->ev_kernel[i], cudaEventDisableTiming));
    }
    s->stage_ready = true;
    return QW_OK;
}

// Host AoS amplitudes <-> device SoA planes in chunks: copy stream and handle stream alternate over two staging buffers.
static int stream_state(qw_sim *s, void *host, bool to_device) {
    int rc = ensure_stage(s);
    if (rc) return rc;
    const Geom &g = s->g;
    const size_t site_bytes = (size_t)g.cdim * s->esize;
    const long long total = g.batch * g.sites;
    const long long per_chunk = (long long)(QW_STAGE_BYTES / site_bytes);
    // the copy stream must not run ahead of work already queued on the handle's stream (and vice versa)
    QW_CUDA(cudaEventRecord(s->ev_kernel[0], s->stream));
    QW_CUDA(cudaStreamWaitEvent(s->copy_stream, s->ev_kernel[0], 0));
    QW_CUDA(cudaEventRecord(s->ev_kernel[1], s->stream));
    int c = 0;
    for (long long first = 0; first < total; first += per_chunk, ++c) {
        const int b = c & 1;
        const long long count = total - first < per_chunk ? total - first : per_chunk;
        char *h = static_cast<char *>(host) + (size_t)first * site_bytes;
        if (to_device) {
            QW_CUDA(cudaStreamWaitEvent(s->copy_stream, s->ev_kernel[b], 0));       // buffer b consumed by chunk c-2
            QW_CUDA(cudaMemcpyAsync(s->stage[b], h, (size_t)count * site_bytes, cudaMemcpyHostToDevice, s->copy_stream));
            QW_CUDA(cudaEventRecord(s->ev_copy[b], s->copy_stream));
            QW_CUDA(cudaStreamWaitEvent(s->stream, s->ev_copy[b], 0));
            rc = launch_aos_to_soa(s, s->stage[b], state_ptr(s, s->cur), first, count);
            if (rc) return rc;
            QW_CUDA(cudaEventRecord(s->ev_kernel[b], s->stream));
        } else {
            QW_CUDA(cudaStreamWaitEvent(s->stream, s->ev_copy[b], 0));              // buffer b copied out by chunk c-2
            rc = launch_soa_to_aos(s, state_ptr(s, s->cur), s->stage[b], first, count);
            if (rc) return rc;
            QW_CUDA(cudaEventRecord(s->ev_kernel[b], s->stream));
            QW_CUDA(cudaStreamWaitEvent(s->copy_stream, s->ev_kernel[b], 0));
            QW_CUDA(cudaMemcpyAsync(h, s->stage[b], (size_t)count * site_bytes, cudaMemcpyDeviceToHost, s->copy_stream));
            QW_CUDA(cudaEventRecord(s->ev_copy[b], s->copy_stream));
        }
    }
    QW_CUDA(cudaStreamSynchronize(s->copy_stream));        // the host buffer is reusable / filled on return
    QW_CUDA(cudaStreamSynchronize(s->stream));
    return QW_OK;
}

// Every call that touches device state must run with the handle's device current: kernels are launched on the current
// device with the handle's pointers, so a mismatch would be a sticky context error instead of a return code.
static int check_device(const qw_sim *s) {
    int dev = -1;
    QW_CUDA(cudaGetDevice(&dev));
    if (dev != s->device)
        return fail(QW_EINVAL, "the handle lives on device %d but device %d is current (cudaSetDevice first)", s->device, dev);
    return QW_OK;
}
#define QW_ON_DEVICE(s) do { int qw_rc_ = check_device(s); if (qw_rc_) return qw_rc_; } while (0)

static int classify_coin(const double *C, int cdim, int dtype) {
    auto re = [&](int a, int b) { return C[2 * (a * cdim + b)]; };
    auto im = [&](int a, int b) { return C[2 * (a * cdim + b) + 1]; };
    bool real = true;
    for (int i = 0; i < cdim * cdim; ++i) if (C[2 * i + 1] != 0.0) real = false;
    if (cdim == 2) {
        const double sv = re(0, 0);
        if (real && sv != 0.0 && re(0, 1) == sv && re(1, 0) == sv && re(1, 1) == -sv) return COIN_HADAMARD;
        return COIN_GENERAL;
    }
    // the 4x4 kinds require a power-of-two overall scale (1/2 for the unitary coins): the temporally blocked kernels
    // defer it, which is exact only then (qw_coin.cuh: apply_coin_bare)
    auto pow2 = [](double x) { int e; const double m = frexp(x < 0 ? -x : x, &e); return m == 0.5; };
    const double h = re(0, 0);
    if (real && h != 0.0 && pow2(h)) {
        static const int sgn[4][4] = {{1, 1, 1, 1}, {1, -1, 1, -1}, {1, 1, -1, -1}, {1, -1, -1, 1}};
        bool hxh = true;
        for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) if (re(a, b) != sgn[a][b] * h) hxh = false;
        if (hxh) return COIN_HXH4;
    }
    if (real) {
        const double d = re(0, 0), g = re(0, 1);
        bool gro = true;
        for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) if (re(a, b) != (a == b ? d : g)) gro = false;
        // the kernel evaluates g*sum + (d-g)*psi_a: only exact when d-g is representable
        bool exact;
        if (dtype == QW_C64) { volatile float dg = (float)d - (float)g; volatile float back = dg + (float)g; exact = (back == (float)d); }
        else                 { volatile double dg = d - g; volatile double back = dg + g; exact = (back == d); }
        if (gro && exact && g != 0.0 && pow2(g)) return COIN_GROVER4;
    }
    if (h != 0.0 && im(0, 0) == 0.0 && pow2(h)) {
        bool dft = true;
        for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
            const int p = (a * b) & 3;
            const double wr = (p == 0) ? h : (p == 2 ? -h : 0.0);
            const double wi = (p == 1) ? h : (p == 3 ? -h : 0.0);
            if (re(a, b) != wr || im(a, b) != wi) dft = false;
        }
        if (dft) return COIN_DFT4;
    }
    return COIN_GENERAL;
}

// Source box of the next step (left = max(mid - extra - it, 1), ...).
// k = 1: the source sites of the next step; k > 1: the sites that can be non-zero after k more steps.
static Box step_box(const qw_sim *s, long long k = 1) {
    const Geom &g = s->g;
    Box b{0, g.em - 1, 0, g.en - 1};
    if (!s->window_enabled || !s->window_valid) return b;
    const long long r = s->radius + k;   // k = 1: pad of one site, like the paper's `extra`
    auto clampdim = [&](long long c, long long ext, long long &lo, long long &hi) {
        long long l = c - r, h = c + r;
        if (g.boundary == QW_PERIODIC) { if (l < 0 || h >= ext) { l = 0; h = ext - 1; } }
        else { if (l < 0) l = 0; if (h >= ext) h = ext - 1; }
        lo = l; hi = h;
    };
    if (g.dim == 1) clampdim(s->centre[0], g.en, b.n_lo, b.n_hi);
    else { clampdim(s->centre[0], g.em, b.m_lo, b.m_hi); clampdim(s->centre[1], g.en, b.n_lo, b.n_hi); }
    return b;
}

}  // namespace qw

using namespace qw;

extern "C" {

const char *qw_last_error(void) { return g_err; }

int qw_create_batch(int64_t batch, int dim, const int64_t *extents, int coin_dim, int dtype, int boundary,
                    qw_sim **out) {
    clear_error();
    if (!out) return fail(QW_EINVAL, "out is NULL");
    *out = nullptr;
    if (!extents) return fail(QW_EINVAL, "extents is NULL");
    if (dim != 1 && dim != 2) return fail(QW_EINVAL, "dim must be 1 or 2 (got %d)", dim);
    if (coin_dim != 2 * dim) return fail(QW_EINVAL, "coin_dim must be 2*dim = %d (got %d)", 2 * dim, coin_dim);
    if (dtype != QW_C64 && dtype != QW_C128) return fail(QW_EINVAL, "dtype must be QW_C64 or QW_C128");
    if (boundary != QW_PERIODIC && boundary != QW_OPEN) return fail(QW_EINVAL, "boundary must be QW_PERIODIC or QW_OPEN");
    if (batch < 1) return fail(QW_EINVAL, "batch must be >= 1");
    for (int d = 0; d < dim; ++d)
        if (extents[d] < 1) return fail(QW_EINVAL, "extents[%d] must be >= 1", d);

    int dev = 0;
    QW_CUDA(cudaGetDevice(&dev));
    int sms = 0;
    QW_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));

    qw_sim *s = new (std::nothrow) qw_sim();
    if (!s) return fail(QW_ENOMEM, "out of host memory");
    memset(s, 0, sizeof(*s));
    Geom &g = s->g;
    g.dim = dim; g.cdim = coin_dim; g.boundary = boundary; g.lattice = QW_NATURAL;
    g.batch = batch;
    g.em = dim == 1 ? 1 : extents[0];
    g.en = dim == 1 ? extents[0] : extents[1];
    if (g.em > (1LL << 40) / g.en) { delete s; return fail(QW_EINVAL, "lattice too large"); }
    g.sites = g.em * g.en;
    s->dtype = dtype;
    s->esize = dtype == QW_C128 ? 16 : 8;
    // row pitch: 128-byte aligned rows when there is more than one row, else 16-byte aligned
    const long long align_elems = ((batch * g.em > 1) ? 128 : 16) / (long long)s->esize;
    g.ghost = dim == 2 ? QW_GHOST_2D : 0;
    g.pitch = (g.en + 2 * g.ghost + align_elems - 1) / align_elems * align_elems;
    g.walk_stride = (g.em + 2 * g.ghost) * g.pitch;
    g.plane_stride = g.batch * g.walk_stride;
    g.origin = (long long)g.ghost * g.pitch + g.ghost;
    s->device = dev; s->sm_count = sms; s->stream = 0;
    s->state_bytes = (size_t)g.cdim * (size_t)g.plane_stride * s->esize;
    s->window_enabled = true;
    s->sched = QW_SCHED_AUTO; s->last_sched = QW_SCHED_AUTO; s->last_k = 1;
    for (int i = 0; i < 2; ++i) {
        cudaError_t e = cudaMalloc(&s->buf[i], s->state_bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            if (i == 1) cudaFree(s->buf[0]);
            const size_t want = s->state_bytes;
            delete s;
            return fail(e == cudaErrorMemoryAllocation ? QW_ENOMEM : QW_ECUDA, "cudaMalloc(%zu) failed: %s",
                        want, cudaGetErrorString(e));
        }
    }
    cudaError_t e = cudaMemset(s->buf[0], 0, s->state_bytes);
    if (e == cudaSuccess) e = cudaMemset(s->buf[1], 0, s->state_bytes);
    if (e != cudaSuccess) {
        cudaFree(s->buf[0]); cudaFree(s->buf[1]); delete s;
        return fail(QW_ECUDA, "cudaMemset failed: %s", cudaGetErrorString(e));
    }
    *out = s;
    return QW_OK;
}

int qw_create(int dim, const int64_t *extents, int coin_dim, int dtype, int boundary, qw_sim **out) {
    return qw_create_batch(1, dim, extents, coin_dim, dtype, boundary, out);
}

int qw_destroy(qw_sim *s) {
    clear_error();
    if (!s) return QW_OK;
    cudaStreamSynchronize(s->stream);
    cudaFree(s->buf[0]); cudaFree(s->buf[1]);
    if (s->d_coin) cudaFree(s->d_coin);
    if (s->d_phases) cudaFree(s->d_phases);
    if (s->d_broken) cudaFree(s->d_broken);
    if (s->scratch) cudaFree(s->scratch);
    if (s->partials) cudaFree(s->partials);
    if (s->stage_ready) {
        cudaStreamSynchronize(s->copy_stream);
        for (int i = 0; i < 2; ++i) { cudaFree(s->stage[i]); cudaEventDestroy(s->ev_copy[i]); cudaEventDestroy(s->ev_kernel[i]); }
        cudaStreamDestroy(s->copy_stream);
    }
    cudaGetLastError();
    delete s;
    return QW_OK;
}

int qw_set_stream(qw_sim *s, void *cuda_stream) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    QW_CUDA(cudaStreamSynchronize(s->stream));   // keep work already issued ordered before the switch
    s->stream = static_cast<cudaStream_t>(cuda_stream);
    return QW_OK;
}

int qw_set_lattice(qw_sim *s, int lattice) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    if (lattice != QW_NATURAL && lattice != QW_DIAGONAL) return fail(QW_EINVAL, "unknown lattice kind %d", lattice);
    if (s->g.dim == 1 && lattice == QW_DIAGONAL) return fail(QW_EINVAL, "the diagonal lattice is 2D only");
    // The light-cone bookkeeping (`radius`: Chebyshev distance, and the L1 diamond the tiled kernel derives from it) counts
    // one axis move per step of the NATURAL lattice; steps taken on the other lattice spread differently, so a change of
    // lattice in mid-walk drops the window (exactness first; qw_set_state_delta re-arms it).
    if (lattice != s->g.lattice && s->has_state && s->t != 0) s->window_valid = false;
    s->g.lattice = lattice;
    return QW_OK;
}

int qw_set_coin(qw_sim *s, int mode, const void *coin) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    if (!coin) return fail(QW_EINVAL, "coin is NULL");
    if (mode != QW_COIN_UNIFORM && mode != QW_COIN_PER_WALK && mode != QW_COIN_PER_SITE)
        return fail(QW_EINVAL, "unknown coin mode %d", mode);
    const Geom &g = s->g;
    const size_t one = (size_t)g.cdim * g.cdim * s->esize;
    if (mode == QW_COIN_UNIFORM) {
        unsigned char tmp[16 * 16];
        if (is_device_ptr(coin)) {
            QW_CUDA(cudaMemcpyAsync(tmp, coin, one, cudaMemcpyDeviceToHost, s->stream));
            QW_CUDA(cudaStreamSynchronize(s->stream));
        } else {
            memcpy(tmp, coin, one);
        }
        for (int i = 0; i < 2 * g.cdim * g.cdim; ++i)
            s->h_coin[i] = s->dtype == QW_C128 ? reinterpret_cast<double *>(tmp)[i] : (double)reinterpret_cast<float *>(tmp)[i];
        s->coin_kind = classify_coin(s->h_coin, g.cdim, s->dtype);
        if (s->d_coin) { QW_CUDA(cudaStreamSynchronize(s->stream)); cudaFree(s->d_coin); s->d_coin = nullptr; }
    } else {
        const size_t count = mode == QW_COIN_PER_WALK ? (size_t)g.batch : (size_t)g.batch * (size_t)g.sites;
        void *d = nullptr;
        cudaError_t e = cudaMalloc(&d, count * one);
        if (e != cudaSuccess) { cudaGetLastError(); return fail(QW_ENOMEM, "cannot allocate %zu bytes for the coin family", count * one); }
        cudaError_t e2 = cudaMemcpyAsync(d, coin, count * one, is_device_ptr(coin) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s->stream);
        if (e2 != cudaSuccess) { cudaFree(d); return fail(QW_ECUDA, "copy of the coin family failed: %s", cudaGetErrorString(e2)); }
        QW_CUDA(cudaStreamSynchronize(s->stream));
        if (s->d_coin) cudaFree(s->d_coin);
        s->d_coin = d;
        s->coin_kind = COIN_GENERAL;
    }
    s->coin_mode = mode;
    s->has_coin = true;
    return QW_OK;
}

int qw_set_site_phases(qw_sim *s, const void *phases) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    QW_CUDA(cudaStreamSynchronize(s->stream));
    if (!phases) { if (s->d_phases) cudaFree(s->d_phases); s->d_phases = nullptr; return QW_OK; }
    const size_t bytes = (size_t)s->g.batch * (size_t)s->g.sites * s->esize;
    void *d = nullptr;
    if (cudaMalloc(&d, bytes) != cudaSuccess) { cudaGetLastError(); return fail(QW_ENOMEM, "cannot allocate %zu bytes for the phases", bytes); }
    cudaError_t e = cudaMemcpyAsync(d, phases, bytes, is_device_ptr(phases) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s->stream);
    if (e != cudaSuccess) { cudaFree(d); return fail(QW_ECUDA, "copy of the phases failed: %s", cudaGetErrorString(e)); }
    QW_CUDA(cudaStreamSynchronize(s->stream));
    if (s->d_phases) cudaFree(s->d_phases);
    s->d_phases = d;
    return QW_OK;
}

int qw_set_broken_links(qw_sim *s, const uint8_t *mask) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    QW_CUDA(cudaStreamSynchronize(s->stream));
    if (!mask) { if (s->d_broken) cudaFree(s->d_broken); s->d_broken = nullptr; return QW_OK; }
    const size_t bytes = (size_t)s->g.batch * (size_t)s->g.sites * (size_t)s->g.cdim;
    void *d = nullptr;
    if (cudaMalloc(&d, bytes) != cudaSuccess) { cudaGetLastError(); return fail(QW_ENOMEM, "cannot allocate %zu bytes for the link mask", bytes); }
    cudaError_t e = cudaMemcpyAsync(d, mask, bytes, is_device_ptr(mask) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s->stream);
    if (e != cudaSuccess) { cudaFree(d); return fail(QW_ECUDA, "copy of the link mask failed: %s", cudaGetErrorString(e)); }
    QW_CUDA(cudaStreamSynchronize(s->stream));
    if (s->d_broken) cudaFree(s->d_broken);
    s->d_broken = static_cast<uint8_t *>(d);
    return QW_OK;
}

int qw_set_random_broken_links(qw_sim *s, int enable, double p, uint64_t seed) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    if (!enable) { s->rbl = false; return QW_OK; }
    if (!(p >= 0.0 && p <= 1.0)) return fail(QW_EINVAL, "the link-breaking probability must lie in [0, 1] (got %g)", p);
    s->rbl = true;
    s->rbl_seed = seed;
    s->rbl_thr = (uint64_t)(p * 4294967296.0);   // floor(p * 2^32): a link is broken iff its 32-bit draw is below it
    return QW_OK;
}

int qw_set_state(qw_sim *s, const void *amps) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    if (!amps) return fail(QW_EINVAL, "amps is NULL");
    const Geom &g = s->g;
    const size_t bytes = (size_t)g.batch * (size_t)g.sites * (size_t)g.cdim * s->esize;
    (void)bytes;
    s->cur = 0;
    if (g.pitch != g.en || g.ghost) QW_CUDA(cudaMemsetAsync(s->buf[0], 0, s->state_bytes, s->stream));
    int rc = is_device_ptr(amps) ? launch_aos_to_soa(s, amps, state_ptr(s, 0))
                                 : stream_state(s, const_cast<void *>(amps), true);   // chunked; host buffer reusable on return
    if (rc) return rc;
    s->has_state = true; s->t = 0; s->window_valid = false;
    return QW_OK;
}

int qw_set_state_delta(qw_sim *s, const int64_t *site, const void *coin_vec) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    if (!site || !coin_vec) return fail(QW_EINVAL, "site or coin_vec is NULL");
    const Geom &g = s->g;
    long long st[2] = {0, 0};
    for (int d = 0; d < g.dim; ++d) {
        const long long ext = (g.dim == 1) ? g.en : (d == 0 ? g.em : g.en);
        if (site[d] < 0 || site[d] >= ext) return fail(QW_EINVAL, "site[%d] = %lld outside [0, %lld)", d, (long long)site[d], ext);
        st[d] = site[d];
    }
    unsigned char tmp[64];
    const size_t vb = (size_t)g.cdim * s->esize;
    if (is_device_ptr(coin_vec)) {
        QW_CUDA(cudaMemcpyAsync(tmp, coin_vec, vb, cudaMemcpyDeviceToHost, s->stream));
        QW_CUDA(cudaStreamSynchronize(s->stream));
    } else {
        memcpy(tmp, coin_vec, vb);
    }
    double cv[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int i = 0; i < 2 * g.cdim; ++i)
        cv[i] = s->dtype == QW_C128 ? reinterpret_cast<double *>(tmp)[i] : (double)reinterpret_cast<float *>(tmp)[i];
    QW_CUDA(cudaMemsetAsync(s->buf[0], 0, s->state_bytes, s->stream));
    QW_CUDA(cudaMemsetAsync(s->buf[1], 0, s->state_bytes, s->stream));
    s->cur = 0;
    int rc = launch_delta(s, st, cv);
    if (rc) return rc;
    s->has_state = true; s->t = 0;
    s->window_valid = true; s->radius = 0;
    s->centre[0] = st[0]; s->centre[1] = st[1];
    return QW_OK;
}

int qw_get_state(const qw_sim *cs, void *amps) {
    clear_error();
    qw_sim *s = const_cast<qw_sim *>(cs);
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    if (!amps) return fail(QW_EINVAL, "amps is NULL");
    if (!s->has_state) return fail(QW_ESTATE, "no state has been set");
    const Geom &g = s->g;
    const size_t bytes = (size_t)g.batch * (size_t)g.sites * (size_t)g.cdim * s->esize;
    (void)bytes;
    if (is_device_ptr(amps)) return launch_soa_to_aos(s, state_ptr(s, s->cur), amps);
    return stream_state(s, amps, false);
}

int qw_step(qw_sim *s, int64_t n) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    if (n < 0) return fail(QW_EINVAL, "n must be >= 0 (got %lld)", (long long)n);
    if (!s->has_coin) return fail(QW_ESTATE, "qw_step before qw_set_coin");
    if (!s->has_state) return fail(QW_ESTATE, "qw_step before qw_set_state");
    if (n == 0) return QW_OK;
    // ---- schedule dispatch (all schedules produce bit-identical states) ----------------------------
    int sched = s->sched;
    if (sched == QW_SCHED_AUTO)
        sched = resident1d_eligible(s) ? QW_SCHED_RESIDENT
              : ((blocked1d_eligible(s) && n >= 4) ||
                 (chain1d_eligible(s, chain1d_granule(s)) && n >= chain1d_granule(s))) ? QW_SCHED_BLOCKED
              : ((tiled2d_eligible(s) || stream2d_eligible(s)) && n >= 2) ? QW_SCHED_TILED : QW_SCHED_FUSED;
    if (sched == QW_SCHED_RESIDENT) {
        if (!resident1d_eligible(s))
            return fail(QW_EUNSUPPORTED, "the resident schedule needs 1D walks of at most 4096 sites, no per-site matrices, no link mask");
        int rc = launch_step_resident1d(s, state_ptr(s, s->cur), state_ptr(s, 1 - s->cur), n);
        if (rc) return rc;
        s->cur ^= 1; s->t += n; s->radius += n;
        s->last_sched = sched; s->last_k = (int)(n > 0x7fffffff ? 0x7fffffff : n);
        return QW_OK;
    }
    if (sched == QW_SCHED_BLOCKED && !blocked1d_eligible(s) && !blocked2d_eligible(s) && !chain1d_eligible(s, chain1d_granule(s)))
        return fail(QW_EUNSUPPORTED, "the temporally blocked schedule needs a uniform coin without phases or link mask on a 1D "
                                     "lattice of >= %d sites or a natural 2D lattice of >= 32 x 32 sites",
                    32 * blocked1d_granule(s));
    if (sched == QW_SCHED_TILED && !tiled2d_eligible(s) && !stream2d_eligible(s))
        return fail(QW_EUNSUPPORTED, "the tiled schedule needs a uniform coin without phases or link mask on a 2D lattice of "
                                     ">= 32 x 32 sites (diagonal lattice: a torus, or an open lattice with a delta start)");
    // natural lattice: the streaming kernel unless the CTA tiles are asked for (which have no instance with link draws)
    const bool stream2d = sched == QW_SCHED_TILED && stream2d_eligible(s) && (s->tiled2d_kernel != 1 || !tiled2d_eligible(s));
    if (sched == QW_SCHED_TILED && (s->sched_k < 0 || s->sched_k % 2 != 0 || s->sched_k > (stream2d ? stream2d_max_k(s) : 8)))
        return fail(QW_EINVAL, "the tiled schedule takes an even k <= %d here (got %d)", stream2d ? stream2d_max_k(s) : 8, s->sched_k);
    int64_t remaining = n;
    s->last_sched = sched; s->last_k = 1;
    if (sched == QW_SCHED_TILED) {
        // k-step launches, then the even part of the remainder; an odd last step goes through the fused kernel below
        // measured optima on B200 (profiles/), both kernels: 8 (complex64) / 6 (complex128); with link draws (integer
        // bound, the draws cost registers) 4
        const int kmax = s->sched_k > 0 ? s->sched_k : (s->rbl ? 4 : (s->dtype == QW_C128 ? 6 : 8));
        s->last_k = kmax;
        while (remaining >= 2) {
            const int kk = (int)(remaining >= kmax ? kmax : remaining / 2 * 2);
            if (!tiled2d_diag_open_ok(s, kk)) break;       // the cone reaches a wall: the fused kernel (which has wall code) takes over
            const Box box = step_box(s, kk);
            int rc = stream2d ? launch_step_stream2d(s, s->cur, 1 - s->cur, kk, box) : launch_step_tiled2d(s, s->cur, 1 - s->cur, kk, box);
            if (rc) return rc;
            s->cur ^= 1; s->t += kk; s->radius += kk; remaining -= kk;
        }
    }
    if (sched == QW_SCHED_BLOCKED && s->g.dim == 2) {
        int kmax = s->sched_k > 0 ? s->sched_k : (s->dtype == QW_C128 ? 4 : 6);   // measured optima (profiles/)
        if (kmax > blocked2d_max_k(s)) kmax = blocked2d_max_k(s);
        s->last_k = kmax;
        while (remaining > 0) {
            const int kk = (int)(remaining >= kmax ? kmax : remaining);
            int rc = launch_step_blocked2d(s, s->cur, 1 - s->cur, kk);
            if (rc) return rc;
            s->touched += (double)s->g.batch * (double)s->g.sites * kk;
            s->cur ^= 1; s->t += kk; s->radius += kk; remaining -= kk;
        }
        return QW_OK;
    }
    if (sched == QW_SCHED_BLOCKED) {
        const int M = blocked1d_granule(s);
        // Halo kernel (qw_step_blocked1d.cu), measured optima on B200 (profiles/r01_blocked1d_v2.md): Hadamard (512-site
        // tiles, 4 FP instr per site-step) k = 48; general coin (256-site tiles, 16 FP instr per site-step: the halo
        // recomputation costs more than the HBM trips) k = 16
        int kmax = s->sched_k > 0 ? s->sched_k : (M == 16 ? 48 : 16);
        // a lattice with fewer tiles than resident warps is launch bound (a launch costs ~50 us whatever k, mostly
        // instruction fetch): take the deepest launches instead
        if (s->sched_k == 0 && s->g.batch * ((s->g.en + (32 * M - 96) - 1) / (32 * M - 96)) < 8LL * s->sm_count)
            kmax = blocked1d_max_k(s);
        if (kmax > blocked1d_max_k(s)) kmax = blocked1d_max_k(s);
        kmax = kmax / M * M;
        if (kmax < M) kmax = M;
        // Chain kernel (qw_step_chain1d.cu; rings): no halo recomputation, one starter tile per chain instead.  Depth:
        // the user's k, else the deepest its FIFO holds.  It is taken whenever it advances a step with fewer tile
        // computations per warp than the halo kernel (always, on lattices of many tiles per warp).
        int kchain = s->sched_k > 0 ? s->sched_k : chain1d_max_k(s);
        if (kchain > chain1d_max_k(s)) kchain = chain1d_max_k(s);
        kchain = kchain / M * M;
        bool chain = kchain >= M && chain1d_eligible(s, kchain);
        const bool halo = blocked1d_eligible(s);       // no random broken links in the halo kernel
        if (chain && halo && s->blocked1d_kernel == 0) chain = chain1d_cost(s, kchain) / kchain < blocked1d_cost(s, kmax) / kmax;
        if (halo && s->blocked1d_kernel == 1) chain = false;
        s->last_k = chain ? kchain : kmax;
        // multiples of M with the big tiles, then a remainder of 4 .. 15 steps with short 8- / 4-step launches (small
        // tiles, the fused kernel's arithmetic), then at most 3 fused single steps
        // (neither kernel applies — e.g. random broken links with a user depth below the tile granule: all steps run fused)
        while ((halo || chain) && remaining >= (halo ? 4 : M)) {
            int rc;
            int kk;
            if (chain && remaining >= M) {
                kk = (int)(remaining >= kchain ? kchain : remaining / M * M);
                rc = launch_step_chain1d(s, state_ptr(s, s->cur), state_ptr(s, 1 - s->cur), kk);
                if (!rc) s->touched += (double)s->g.batch * (double)s->g.sites * kk;
            } else {
                kk = remaining >= M ? (int)(remaining >= kmax ? kmax : remaining / M * M) : (remaining >= 8 ? 8 : 4);
                rc = launch_step_blocked1d(s, state_ptr(s, s->cur), state_ptr(s, 1 - s->cur), kk);
                if (!rc) s->touched += (double)s->g.batch * (double)s->g.sites * kk;
            }
            if (rc) return rc;
            s->cur ^= 1; s->t += kk; s->radius += kk; remaining -= kk;
        }
    }
    const bool allow_fast = sched != QW_SCHED_GENERIC;
    for (int64_t i = 0; i < remaining; ++i) {
        const Box box = step_box(s);
        int rc = launch_step(s, state_ptr(s, s->cur), state_ptr(s, 1 - s->cur), box, allow_fast);
        if (rc) return rc;
        s->touched += (double)s->g.batch * (double)(box.m_hi - box.m_lo + 1) * (double)(box.n_hi - box.n_lo + 1);
        s->cur ^= 1; s->t += 1; s->radius += 1;
    }
    return QW_OK;
}

int qw_step_inverse(qw_sim *s, int64_t n) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    if (n < 0) return fail(QW_EINVAL, "n must be >= 0 (got %lld)", (long long)n);
    if (!s->has_coin) return fail(QW_ESTATE, "qw_step_inverse before qw_set_coin");
    if (!s->has_state) return fail(QW_ESTATE, "qw_step_inverse before qw_set_state");
    if (s->rbl && n > s->t)
        return fail(QW_ESTATE, "with random broken links U(t) is defined for t >= 0 only: cannot take %lld inverse steps at t = %lld",
                    (long long)n, s->t);
    for (int64_t i = 0; i < n; ++i) {
        int rc = launch_step_inverse(s, state_ptr(s, s->cur), state_ptr(s, 1 - s->cur));
        if (rc) return rc;
        s->cur ^= 1; s->t -= 1; s->radius += 1;
    }
    return QW_OK;
}

int qw_probabilities(const qw_sim *cs, void *out) {
    clear_error();
    qw_sim *s = const_cast<qw_sim *>(cs);
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    if (!out) return fail(QW_EINVAL, "out is NULL");
    if (!s->has_state) return fail(QW_ESTATE, "no state has been set");
    const size_t bytes = (size_t)s->g.batch * (size_t)s->g.sites * (s->esize / 2);
    if (is_device_ptr(out)) return launch_probabilities(s, state_ptr(s, s->cur), out);
    int rc = ensure_scratch(s, bytes);
    if (rc) return rc;
    rc = launch_probabilities(s, state_ptr(s, s->cur), s->scratch);
    if (rc) return rc;
    QW_CUDA(cudaMemcpyAsync(out, s->scratch, bytes, cudaMemcpyDeviceToHost, s->stream));
    QW_CUDA(cudaStreamSynchronize(s->stream));
    return QW_OK;
}

int qw_probabilities_mean(const qw_sim *cs, void *out) {
    clear_error();
    qw_sim *s = const_cast<qw_sim *>(cs);
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    if (!out) return fail(QW_EINVAL, "out is NULL");
    if (!s->has_state) return fail(QW_ESTATE, "no state has been set");
    const size_t bytes = (size_t)s->g.sites * (s->esize / 2);
    if (is_device_ptr(out)) return launch_probabilities_mean(s, state_ptr(s, s->cur), out);
    int rc = ensure_scratch(s, bytes);
    if (rc) return rc;
    rc = launch_probabilities_mean(s, state_ptr(s, s->cur), s->scratch);
    if (rc) return rc;
    QW_CUDA(cudaMemcpyAsync(out, s->scratch, bytes, cudaMemcpyDeviceToHost, s->stream));
    QW_CUDA(cudaStreamSynchronize(s->stream));
    return QW_OK;
}

int qw_moments(const qw_sim *cs, double *out) {
    clear_error();
    qw_sim *s = const_cast<qw_sim *>(cs);
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    if (!out) return fail(QW_EINVAL, "out is NULL");
    if (!s->has_state) return fail(QW_ESTATE, "no state has been set");
    const size_t bytes = (size_t)s->g.batch * (s->g.dim == 1 ? 3 : 6) * sizeof(double);
    if (is_device_ptr(out)) return launch_moments(s, state_ptr(s, s->cur), out);
    int rc = ensure_scratch(s, bytes);
    if (rc) return rc;
    rc = launch_moments(s, state_ptr(s, s->cur), static_cast<double *>(s->scratch));
    if (rc) return rc;
    QW_CUDA(cudaMemcpyAsync(out, s->scratch, bytes, cudaMemcpyDeviceToHost, s->stream));
    QW_CUDA(cudaStreamSynchronize(s->stream));
    return QW_OK;
}

int qw_moments_static(const qw_sim *cs, double *out) {
    clear_error();
    qw_sim *s = const_cast<qw_sim *>(cs);
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_ON_DEVICE(s);
    if (!out) return fail(QW_EINVAL, "out is NULL");
    if (!s->has_state) return fail(QW_ESTATE, "no state has been set");
    if (!is_device_ptr(out)) return fail(QW_EINVAL, "qw_moments_static writes to DEVICE memory only (a host buffer would need a staging allocation)");
    return launch_moments_static(s, state_ptr(s, s->cur), out);
}

int qw_set_schedule(qw_sim *s, int schedule, int k) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    if (schedule < QW_SCHED_AUTO || schedule > QW_SCHED_TILED) return fail(QW_EINVAL, "unknown schedule %d", schedule);
    if (k < 0) return fail(QW_EINVAL, "k must be >= 0");
    s->sched = schedule; s->sched_k = k;
    return QW_OK;
}

int qw_set_option(qw_sim *s, int key, int64_t value) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    switch (key) {
        case QW_OPT_MAX_CTAS:
            if (value < 0 || value > 0x7fffffff) return fail(QW_EINVAL, "QW_OPT_MAX_CTAS must be >= 0");
            s->max_ctas = (int)value;
            break;
        case QW_OPT_BLOCKED1D_KERNEL:
            if (value < 0 || value > 2) return fail(QW_EINVAL, "QW_OPT_BLOCKED1D_KERNEL must be 0 (auto), 1 (halo tiles) or 2 (chained tiles)");
            s->blocked1d_kernel = (int)value;
            break;
        case QW_OPT_TILED2D_KERNEL:
            if (value < 0 || value > 2) return fail(QW_EINVAL, "QW_OPT_TILED2D_KERNEL must be 0 (auto), 1 (CTA tiles) or 2 (streaming warps)");
            s->tiled2d_kernel = (int)value;
            break;
        default: return fail(QW_EINVAL, "unknown option key %d", key);
    }
    return QW_OK;
}

int qw_set_window(qw_sim *s, int enable) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    s->window_enabled = enable != 0;
    return QW_OK;
}

int qw_get_info(const qw_sim *s, int what, int64_t *out) {
    clear_error();
    if (!s || !out) return fail(QW_EINVAL, "NULL argument");
    switch (what) {
        case QW_INFO_LAUNCHES: *out = s->launches; break;
        case QW_INFO_TIME: *out = s->t; break;
        case QW_INFO_LAST_SCHEDULE: *out = s->last_sched; break;
        case QW_INFO_LAST_K: *out = s->last_k; break;
        case QW_INFO_STATE_BYTES: *out = (int64_t)s->state_bytes; break;
        case QW_INFO_WINDOW: *out = (s->window_enabled && s->window_valid) ? 1 : 0; break;
        case QW_INFO_SITES_TOUCHED: *out = (int64_t)s->touched; break;
        default: return fail(QW_EINVAL, "unknown info key %d", what);
    }
    return QW_OK;
}

int qw_synchronize(const qw_sim *s) {
    clear_error();
    if (!s) return fail(QW_EINVAL, "handle is NULL");
    QW_CUDA(cudaStreamSynchronize(s->stream));
    return QW_OK;
}

}  // extern "C"
