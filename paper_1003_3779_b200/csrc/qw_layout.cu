// qw_layout.cu — layout kernels off the timed path: user-side AoS [walk][site][coin] <-> device
// SoA plane[coin][walk][m][n_pitch], and the delta start
// |site> (x) coin_vec of PAPER.md:126-134 (every figure of the paper starts from one site).
#include "qw_coin.cuh"

namespace qw {

constexpr int LAYOUT_BLOCK = 256;

template <typename R, int CD, bool TO_SOA>
__global__ void __launch_bounds__(LAYOUT_BLOCK)
transpose_kernel(const typename Cx<R>::T *__restrict__ src, typename Cx<R>::T *__restrict__ dst,
                 long long first, long long count, long long sites, long long en, long long pitch,
                 long long walk_stride, long long plane_stride) {
    // the AoS side holds the flat sites [first, first + count) (flat = walk * sites + site), starting at its element 0
    const long long j = (long long)blockIdx.x * LAYOUT_BLOCK + threadIdx.x;
    if (j >= count) return;
    const long long i = first + j;
    const long long w = i / sites, x = i - w * sites;
    const long long m = x / en, n = x - m * en;
    const long long idx = w * walk_stride + m * pitch + n;
#pragma unroll
    for (int c = 0; c < CD; ++c) {
        if (TO_SOA) dst[c * plane_stride + idx] = src[j * CD + c];
        else        dst[j * CD + c] = src[c * plane_stride + idx];
    }
}

template <typename R, int CD, bool TO_SOA>
static int launch_transpose_t(qw_sim *s, const void *src, void *dst, long long first, long long count) {
    typedef typename Cx<R>::T V;
    const Geom &g = s->g;
    const long long blocks = (count + LAYOUT_BLOCK - 1) / LAYOUT_BLOCK;
    if (blocks <= 0) return QW_OK;
    if (blocks > 0x7fffffffLL) return fail(QW_EUNSUPPORTED, "lattice too large for one launch");
    transpose_kernel<R, CD, TO_SOA><<<(unsigned)blocks, LAYOUT_BLOCK, 0, s->stream>>>(
        static_cast<const V *>(src), static_cast<V *>(dst), first, count, g.sites, g.en, g.pitch,
        g.walk_stride, g.plane_stride);
    QW_LAUNCH_CHECK(s, "transpose_kernel");
    return QW_OK;
}

// `aos` points at the amplitudes of flat site `first`; count < 0 = all sites of all walks
int launch_aos_to_soa(qw_sim *s, const void *aos, void *soa, long long first, long long count) {
    if (count < 0) count = s->g.batch * s->g.sites - first;
    if (s->dtype == QW_C128)
        return s->g.cdim == 2 ? launch_transpose_t<double, 2, true>(s, aos, soa, first, count)
                              : launch_transpose_t<double, 4, true>(s, aos, soa, first, count);
    return s->g.cdim == 2 ? launch_transpose_t<float, 2, true>(s, aos, soa, first, count)
                          : launch_transpose_t<float, 4, true>(s, aos, soa, first, count);
}

int launch_soa_to_aos(qw_sim *s, const void *soa, void *aos, long long first, long long count) {
    if (count < 0) count = s->g.batch * s->g.sites - first;
    if (s->dtype == QW_C128)
        return s->g.cdim == 2 ? launch_transpose_t<double, 2, false>(s, soa, aos, first, count)
                              : launch_transpose_t<double, 4, false>(s, soa, aos, first, count);
    return s->g.cdim == 2 ? launch_transpose_t<float, 2, false>(s, soa, aos, first, count)
                          : launch_transpose_t<float, 4, false>(s, soa, aos, first, count);
}

template <typename R>
__global__ void delta_kernel(typename Cx<R>::T *soa, long long batch, int cdim, long long walk_stride,
                             long long plane_stride, long long offset, const double4 v01, const double4 v23) {
    const long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= batch) return;
    const double vals[8] = {v01.x, v01.y, v01.z, v01.w, v23.x, v23.y, v23.z, v23.w};
    for (int c = 0; c < cdim; ++c) {
        typename Cx<R>::T z; z.x = (R)vals[2 * c]; z.y = (R)vals[2 * c + 1];
        soa[c * plane_stride + w * walk_stride + offset] = z;
    }
}

// Caller has zeroed the buffer.  coin_vec: cdim complex promoted to double (exact for float input).
int launch_delta(qw_sim *s, const long long *site, const double *cv) {
    const Geom &g = s->g;
    const long long off = (g.dim == 1) ? site[0] : site[0] * g.pitch + site[1];
    double4 a = make_double4(cv[0], cv[1], cv[2], cv[3]);
    double4 b = g.cdim == 4 ? make_double4(cv[4], cv[5], cv[6], cv[7]) : make_double4(0, 0, 0, 0);
    const unsigned blocks = (unsigned)((g.batch + 127) / 128);
    if (s->dtype == QW_C128)
        delta_kernel<double><<<blocks, 128, 0, s->stream>>>(static_cast<double2 *>(state_ptr(s, s->cur)), g.batch,
                                                             g.cdim, g.walk_stride, g.plane_stride, off, a, b);
    else
        delta_kernel<float><<<blocks, 128, 0, s->stream>>>(static_cast<float2 *>(state_ptr(s, s->cur)), g.batch,
                                                            g.cdim, g.walk_stride, g.plane_stride, off, a, b);
    QW_LAUNCH_CHECK(s, "delta_kernel");
    return QW_OK;
}

}  // namespace qw
