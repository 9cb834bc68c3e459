// qw_step.cu — one-launch-per-step kernels: the fused coin + conditional-shift step
// psi' = S (I (x) C) psi (PAPER.md:42 eq. 2, :80 eq. 7) in SCATTER form: the thread that owns
// source site x applies the coin in registers (eq. 1) and writes every component straight into
// its neighbour site of the other ping-pong buffer (eq. 3 / eq. 8); components whose link is
// broken or leaves an open lattice are written back to x with the opposite coin (eqs. 9-10).
// Each amplitude is read once and written once: 2 * coin_dim * sizeof(complex) bytes per site.
//
// Two instantiation families share the code:
//   FAST    uniform coin held in the kernel parameters (constant bank), no phases, no link
//           mask; natural or diagonal lattice, optional random broken links; U sites per thread, strided by the block so that every warp
//           access is one contiguous run                       -> QW_SCHED_FUSED
//   GENERAL every feature decided at run time (per-walk / per-site coins, phases, broken links,
//           diagonal lattice)                                  -> QW_SCHED_GENERIC
// plus the inverse step U^dagger in gather form (qw_step_inverse).
#include "qw_coin.cuh"
#include "qw_philox.cuh"

namespace qw {

template <typename R, int CD>
struct StepArgs {
    const typename Cx<R>::T *in;
    typename Cx<R>::T *out;
    long long em, en, pitch, walk_stride, plane_stride, sites;
    long long m_lo, n_lo;        // origin of the source box
    long long box_m, box_n;      // extent of the source box
    int chunks_per_row;          // blocks along n
    int boundary, lattice, coin_mode;
    const typename Cx<R>::T *coins;
    const typename Cx<R>::T *phases;
    const uint8_t *broken;
    // random broken links redrawn every step (qw_set_random_broken_links): a link is broken iff
    // philox4x32_10(counter = (owner lo, owner hi, t, walk), key = seed)[axis] < rbl_thr
    int rbl;
    unsigned rbl_key0, rbl_key1;
    unsigned long long rbl_thr;  // floor(p * 2^32), 0 .. 2^32
    unsigned t;                  // step index (low 32 bits) of the U(t) being applied
    R coin[2 * CD * CD];
};

constexpr int STEP_BLOCK = 256;
// Launch shape of the fused kernel, measured on B200 (profiles/r01_fused_step.md, "launch shapes"):
// threads per block BS and sites per thread U (strided by the block).
template <typename R, int DIM> struct FusedShape {
    static constexpr int BS = (DIM == 2 && sizeof(R) == 4) ? 128 : 256;
    static constexpr int U = (DIM == 1) ? (sizeof(R) == 8 ? 4 : 8) : (sizeof(R) == 8 ? 1 : 4);
};

// Is the link that component c of site (m,n) of walk w points along — it ends at (tm,tn) inside the lattice — broken
// at step a.t?  The link is named by its OWNER (the end from which it points in the positive direction: dm > 0, or
// dm = 0 and dn > 0) and its axis (0: along n / along (+1,+1); 1: along m / along (+1,-1)), so that both ends of a
// link evaluate the same function and U(t) stays unitary (eq. 9: RBL is a property of the link).
template <int DIM_LINKS, typename A>
__device__ __forceinline__ bool rbl_link_broken(const A &a, long long w, long long m, long long n, long long tm,
                                                long long tn, int dm, int dn) {
    const bool positive = dm > 0 || (dm == 0 && dn > 0);
    const unsigned long long owner = (unsigned long long)(positive ? (m * a.en + n) : (tm * a.en + tn));
    const int axis = (dm != 0 && dn != 0) ? ((dm * dn > 0) ? 0 : 1) : (dm != 0 ? 1 : 0);
    const unsigned word = rbl_link_word(owner * (DIM_LINKS) + (unsigned)axis, a.t, (unsigned)w, a.rbl_key0, a.rbl_key1);
    return (unsigned long long)word < a.rbl_thr;
}

// FAM (with FAST): the coin FAMILY of PAPER.md:35-38 eq. 1 on the vectorised path — a per-walk matrix (read once per
// thread: all sites of a block belong to one walk) and / or the per-site phase table as a third, coalesced read stream.
template <typename R, int DIM, int KIND, bool FAST, int U, bool RBL = false, int BS = STEP_BLOCK, bool DIAG = false, bool FAM = false>
__global__ void __launch_bounds__(BS)
step_scatter_kernel(const StepArgs<R, 2 * DIM> a) {
    constexpr int CD = 2 * DIM;
    typedef typename Cx<R>::T V;
    // block -> (walk, row m, chunk along n)
    const long long blk = blockIdx.x;
    const long long rowid = blk / a.chunks_per_row;
    const int chunk = (int)(blk - rowid * a.chunks_per_row);
    const long long w = rowid / a.box_m;
    const long long m = a.m_lo + (rowid - w * a.box_m);
    const long long n_base = (long long)chunk * (BS * U) + threadIdx.x;
    const long long row_off = w * a.walk_stride + m * a.pitch;

    cplx<R> v[U][CD];
    bool live[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const long long nb = n_base + (long long)u * BS;
        live[u] = nb < a.box_n;
        if (live[u]) {
            const long long idx = row_off + a.n_lo + nb;
#pragma unroll
            for (int b = 0; b < CD; ++b) v[u][b] = cx_load<R>(a.in + b * a.plane_stride + idx);
        }
    }
    // Random broken links on the natural lattice / in 1D: every site evaluates the ONE Philox call it owns (links to
    // n+1 and to m+1); the link to n-1 is the left neighbour's: it comes through shared memory (the block's sites
    // are consecutive along n), only the first site of a block recomputes it.  The link to m-1 belongs to another
    // block's row and is recomputed.  2 -> 1 calls per site in 1D, 3 -> 2 in 2D.
    constexpr bool SHARE = FAST && RBL && !DIAG;
    __shared__ unsigned char link_n[SHARE ? U : 1][SHARE ? BS : 1];
    unsigned own[U];
    if constexpr (SHARE && DIM == 1 && U % 4 == 0) {
        // 1D: one generator call serves FOUR consecutive sites (reading R27), and for each u the lanes 4q .. 4q+3 of a
        // warp hold four consecutive sites.  So for every group of four u's, lane l evaluates the call(s) of ONE quad —
        // row u = ub + (l & 3), quad q = l >> 2 — and the lanes fetch their bit with a shuffle: U/4 calls per thread
        // instead of U (twice that when the window starts at a site that is not a multiple of 4).
        const int lane = threadIdx.x & 31;
        const long long wbase = a.n_lo + (long long)chunk * (BS * U) + (threadIdx.x & ~31);   // site of lane 0 at u = 0
        const unsigned r = (unsigned)wbase & 3u;                                               // warp-uniform: BS % 4 == 0
#pragma unroll
        for (int ub = 0; ub < U; ub += 4) {
            const unsigned long long x4 = (unsigned long long)(wbase + (long long)(ub + (lane & 3)) * BS + 4 * (lane >> 2));
            unsigned wd[4];
            rbl_group_words(x4 >> 2, a.t, (unsigned)w, a.rbl_key0, a.rbl_key1, wd);
            unsigned bits = 0;
#pragma unroll
            for (int i = 0; i < 4; ++i) bits |= ((unsigned long long)wd[i] < a.rbl_thr ? 1u : 0u) << i;
            if (r != 0) {
                rbl_group_words((x4 >> 2) + 1, a.t, (unsigned)w, a.rbl_key0, a.rbl_key1, wd);
#pragma unroll
                for (int i = 0; i < 4; ++i) bits |= ((unsigned long long)wd[i] < a.rbl_thr ? 1u : 0u) << (4 + i);
            }
            const unsigned nibble = (bits >> r) & 0xfu;            // sites x4 .. x4+3
#pragma unroll
            for (int du = 0; du < 4; ++du) {
                const unsigned nib = __shfl_sync(0xffffffffu, nibble, 4 * (lane >> 2) + du);
                own[ub + du] = (nib >> (lane & 3)) & 1u;
                link_n[ub + du][threadIdx.x] = (unsigned char)own[ub + du];
            }
        }
        __syncthreads();
    } else if constexpr (SHARE) {
        // 2D, even row length and an even first column (the launcher extends the box by one site if needed): the lanes
        // 2q, 2q+1 hold the two sites of one generator group, so the EVEN lane evaluates the call of the pair's own links
        // and the ODD lane the call of the pair's upper-row links (owners (m-1, n), (m-1, n+1): numbers 2o'+1, 2o'+3 of
        // group o'/2); two shuffles hand the bits out.  One call per site instead of two.
        const bool coop = DIM == 2 && ((a.en & 1) == 0) && ((a.n_lo & 1) == 0);
#pragma unroll
        for (int u = 0; u < U; ++u) {
            own[u] = 0;
            if (coop) {
                const int lane = threadIdx.x & 31;
                const long long nl = a.n_lo + n_base + (long long)u * BS;            // parity of nl = parity of the lane
                unsigned long long grp;
                if ((lane & 1) == 0) {
                    grp = (unsigned long long)(m * a.en + nl) >> 1;
                } else {
                    long long mu = m - 1;
                    if (mu < 0) mu += a.em;
                    grp = (unsigned long long)(mu * a.en + nl - 1) >> 1;
                }
                unsigned wd[4];
                rbl_group_words(grp, a.t, (unsigned)w, a.rbl_key0, a.rbl_key1, wd);
                unsigned pack = 0;
#pragma unroll
                for (int i = 0; i < 4; ++i) pack |= ((unsigned long long)wd[i] < a.rbl_thr ? 1u : 0u) << i;
                const unsigned ownpack = __shfl_sync(0xffffffffu, pack, lane & ~1);
                const unsigned uppack = __shfl_sync(0xffffffffu, pack, lane | 1);
                const unsigned mine = (lane & 1) ? (ownpack >> 2) & 3u : ownpack & 3u;   // bit 0: own n-link, bit 1: own m-link
                const unsigned up = (lane & 1) ? (uppack >> 3) & 1u : (uppack >> 1) & 1u; // words 3 / 1: the upper row's m-links
                own[u] = mine | (up << 2) | 8u;
            } else if (live[u]) {
                // the links this site owns: numbers owner * DIM + axis (1D: word owner & 3 of call owner / 4; 2D: words
                // 2 (owner & 1) + axis of call owner / 2)
                const unsigned long long owner = (unsigned long long)(m * a.en + a.n_lo + n_base + (long long)u * BS);
                unsigned wd[4];
                rbl_group_words((owner * DIM) >> 2, a.t, (unsigned)w, a.rbl_key0, a.rbl_key1, wd);
                unsigned w0, w1;
                if constexpr (DIM == 1) {
                    const unsigned sel = (unsigned)owner & 3u;
                    w0 = sel == 0 ? wd[0] : (sel == 1 ? wd[1] : (sel == 2 ? wd[2] : wd[3]));
                    w1 = 0xffffffffu;                        // no second axis in 1D
                } else {
                    const bool odd = ((unsigned)owner & 1u) != 0;
                    w0 = odd ? wd[2] : wd[0];
                    w1 = odd ? wd[3] : wd[1];
                }
                own[u] = ((unsigned long long)w0 < a.rbl_thr ? 1u : 0u) | ((unsigned long long)w1 < a.rbl_thr ? 2u : 0u);
            }
            link_n[u][threadIdx.x] = (unsigned char)(own[u] & 1u);
        }
        __syncthreads();
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
        if (!live[u]) continue;
        const long long n = a.n_lo + n_base + (long long)u * BS;
        const long long x = m * a.en + n;
        if constexpr (FAST && FAM) {
            if (a.coin_mode == QW_COIN_PER_WALK) {
                const R *Cg = reinterpret_cast<const R *>(a.coins + w * (CD * CD));
                R C[2 * CD * CD];
#pragma unroll
                for (int i = 0; i < 2 * CD * CD; ++i) C[i] = Cg[i];
                apply_coin<R, CD, COIN_GENERAL>(C, v[u]);
            } else {
                apply_coin<R, CD, KIND>(a.coin, v[u]);
            }
            if (a.phases) {
                const cplx<R> ph = cx_load<R>(a.phases + w * a.sites + x);
#pragma unroll
                for (int c = 0; c < CD; ++c) v[u][c] = cx_mul(ph.re, ph.im, v[u][c]);
            }
        } else if constexpr (FAST) {
            apply_coin<R, CD, KIND>(a.coin, v[u]);
        } else {
            if (a.coin_mode == QW_COIN_UNIFORM) {
                apply_coin<R, CD, KIND>(a.coin, v[u]);
            } else {
                const long long ci = (a.coin_mode == QW_COIN_PER_WALK) ? w : (w * a.sites + x);
                const R *Cg = reinterpret_cast<const R *>(a.coins + ci * (CD * CD));
                R C[2 * CD * CD];
#pragma unroll
                for (int i = 0; i < 2 * CD * CD; ++i) C[i] = Cg[i];
                apply_coin<R, CD, COIN_GENERAL>(C, v[u]);
            }
            if (a.phases) {
                const cplx<R> ph = cx_load<R>(a.phases + w * a.sites + x);
#pragma unroll
                for (int c = 0; c < CD; ++c) v[u][c] = cx_mul(ph.re, ph.im, v[u][c]);
            }
        }
#pragma unroll
        for (int c = 0; c < CD; ++c) {
            int dm, dn;
            coin_direction<DIM>(FAST ? (DIAG ? QW_DIAGONAL : QW_NATURAL) : a.lattice, c, dm, dn);
            long long tm = m + dm, tn = n + dn;
            bool stay = false;
            if (a.boundary == QW_PERIODIC) {
                if (DIM == 2) { if (tm < 0) tm += a.em; else if (tm >= a.em) tm -= a.em; }
                if (tn < 0) tn += a.en; else if (tn >= a.en) tn -= a.en;
            } else {
                stay = (tn < 0) | (tn >= a.en);
                if (DIM == 2) stay |= (tm < 0) | (tm >= a.em);
            }
            if constexpr (!FAST) {
                if (a.broken && a.broken[(w * a.sites + x) * CD + c]) stay = true;
                if (a.rbl && !stay && rbl_link_broken<DIM>(a, w, m, n, tm, tn, dm, dn)) stay = true;
            } else if constexpr (SHARE) {
                if (!stay) {
                    bool broken;
                    if (dm == 0 && dn > 0) broken = (own[u] & 1u) != 0;                    // own link along n
                    else if (dm > 0) broken = (own[u] & 2u) != 0;                          // own link along m
                    else if (dm == 0) {                                                    // the left neighbour's link
                        if (threadIdx.x > 0) broken = link_n[u][threadIdx.x - 1] != 0;
                        else if (u > 0) broken = link_n[u > 0 ? u - 1 : 0][BS - 1] != 0;
                        else broken = rbl_link_broken<DIM>(a, w, m, n, tm, tn, dm, dn);         // first site of the block
                    } else broken = (own[u] & 8u) ? (own[u] & 4u) != 0                          // the upper row's link
                                                  : rbl_link_broken<DIM>(a, w, m, n, tm, tn, dm, dn);
                    if (broken) stay = true;
                }
            } else if constexpr (RBL) {
                if (!stay && rbl_link_broken<DIM>(a, w, m, n, tm, tn, dm, dn)) stay = true;
            }
            const long long dst = stay ? ((CD - 1 - c) * a.plane_stride + row_off + n)
                                       : (c * a.plane_stride + w * a.walk_stride + tm * a.pitch + tn);
            cx_store<R>(a.out + dst, v[u][c]);
        }
    }
}

// U^dagger = (I (x) C^dagger) S^dagger in gather form: the thread that owns site x reads back every
// component from where the forward step wrote it, then applies C_x^dagger.
template <typename R, int DIM>
__global__ void __launch_bounds__(STEP_BLOCK)
step_inverse_kernel(const StepArgs<R, 2 * DIM> a) {
    constexpr int CD = 2 * DIM;
    const long long blk = blockIdx.x;
    const long long rowid = blk / a.chunks_per_row;
    const int chunk = (int)(blk - rowid * a.chunks_per_row);
    const long long w = rowid / a.em;
    const long long m = rowid - w * a.em;
    const long long n = (long long)chunk * STEP_BLOCK + threadIdx.x;
    if (n >= a.en) return;
    const long long x = m * a.en + n;
    const long long row_off = w * a.walk_stride + m * a.pitch;
    cplx<R> v[CD];
#pragma unroll
    for (int c = 0; c < CD; ++c) {
        int dm, dn;
        coin_direction<DIM>(a.lattice, c, dm, dn);
        long long tm = m + dm, tn = n + dn;
        bool stay = false;
        if (a.boundary == QW_PERIODIC) {
            if (DIM == 2) { if (tm < 0) tm += a.em; else if (tm >= a.em) tm -= a.em; }
            if (tn < 0) tn += a.en; else if (tn >= a.en) tn -= a.en;
        } else {
            stay = (tn < 0) | (tn >= a.en);
            if (DIM == 2) stay |= (tm < 0) | (tm >= a.em);
        }
        if (a.broken && a.broken[(w * a.sites + x) * CD + c]) stay = true;
        if (a.rbl && !stay && rbl_link_broken<DIM>(a, w, m, n, tm, tn, dm, dn)) stay = true;
        const long long src = stay ? ((CD - 1 - c) * a.plane_stride + row_off + n)
                                   : (c * a.plane_stride + w * a.walk_stride + tm * a.pitch + tn);
        v[c] = cx_load<R>(a.in + src);
    }
    if (a.phases) {   // (ph * C)^dagger = conj(ph) * C^dagger
        const cplx<R> ph = cx_load<R>(a.phases + w * a.sites + x);
#pragma unroll
        for (int c = 0; c < CD; ++c) v[c] = cx_mul(ph.re, -ph.im, v[c]);
    }
    R C[2 * CD * CD];
    if (a.coin_mode == QW_COIN_UNIFORM) {
#pragma unroll
        for (int i = 0; i < 2 * CD * CD; ++i) C[i] = a.coin[i];
    } else {
        const long long ci = (a.coin_mode == QW_COIN_PER_WALK) ? w : (w * a.sites + x);
        const R *Cg = reinterpret_cast<const R *>(a.coins + ci * (CD * CD));
#pragma unroll
        for (int i = 0; i < 2 * CD * CD; ++i) C[i] = Cg[i];
    }
    apply_coin_dagger<R, CD>(C, v);
#pragma unroll
    for (int b = 0; b < CD; ++b) cx_store<R>(a.out + b * a.plane_stride + row_off + n, v[b]);
}

template <typename R, int DIM>
static void fill_args(const qw_sim *s, const void *in, void *out, const Box &box, StepArgs<R, 2 * DIM> &a) {
    typedef typename Cx<R>::T V;
    const Geom &g = s->g;
    a.in = static_cast<const V *>(in);
    a.out = static_cast<V *>(out);
    a.em = g.em; a.en = g.en; a.pitch = g.pitch; a.walk_stride = g.walk_stride;
    a.plane_stride = g.plane_stride; a.sites = g.sites;
    a.m_lo = box.m_lo; a.n_lo = box.n_lo;
    a.box_m = box.m_hi - box.m_lo + 1; a.box_n = box.n_hi - box.n_lo + 1;
    a.boundary = g.boundary; a.lattice = g.lattice; a.coin_mode = s->coin_mode;
    a.coins = static_cast<const V *>(s->d_coin);
    a.phases = static_cast<const V *>(s->d_phases);
    a.broken = s->d_broken;
    a.rbl = s->rbl ? 1 : 0;
    a.rbl_key0 = (unsigned)(s->rbl_seed & 0xffffffffu); a.rbl_key1 = (unsigned)(s->rbl_seed >> 32);
    a.rbl_thr = s->rbl_thr;
    a.t = (unsigned)((unsigned long long)s->t & 0xffffffffu);
    for (int i = 0; i < 2 * g.cdim * g.cdim; ++i) a.coin[i] = (R)s->h_coin[i];
}

template <typename R, int DIM, int KIND, bool FAST, int U, bool RBL = false, int BS = STEP_BLOCK, bool DIAG = false, bool FAM = false>
static int launch_scatter(qw_sim *s, StepArgs<R, 2 * DIM> &a) {
    const long long per_block = (long long)BS * U;
    a.chunks_per_row = (int)((a.box_n + per_block - 1) / per_block);
    const long long blocks = s->g.batch * a.box_m * a.chunks_per_row;
    if (blocks <= 0) return QW_OK;
    if (blocks > 0x7fffffffLL) return fail(QW_EUNSUPPORTED, "lattice too large for one launch");
    step_scatter_kernel<R, DIM, KIND, FAST, U, RBL, BS, DIAG, FAM><<<(unsigned)blocks, BS, 0, s->stream>>>(a);
    QW_LAUNCH_CHECK(s, "step_scatter_kernel");
    return QW_OK;
}

template <typename R, int DIM, bool RBL, bool DIAG>
static int launch_fast_t(qw_sim *s, StepArgs<R, 2 * DIM> &a) {
    constexpr int UF = FusedShape<R, DIM>::U, BS = FusedShape<R, DIM>::BS;
    switch (s->coin_kind) {
        case COIN_HADAMARD: if (DIM == 1) return launch_scatter<R, DIM, COIN_HADAMARD, true, UF, RBL, BS, DIAG>(s, a); break;
        case COIN_GROVER4:  if (DIM == 2) return launch_scatter<R, DIM, COIN_GROVER4, true, UF, RBL, BS, DIAG>(s, a); break;
        case COIN_HXH4:     if (DIM == 2) return launch_scatter<R, DIM, COIN_HXH4, true, UF, RBL, BS, DIAG>(s, a); break;
        case COIN_DFT4:     if (DIM == 2) return launch_scatter<R, DIM, COIN_DFT4, true, UF, RBL, BS, DIAG>(s, a); break;
        default: break;
    }
    return launch_scatter<R, DIM, COIN_GENERAL, true, UF, RBL, BS, DIAG>(s, a);
}

template <typename R, int DIM>
static int launch_step_t(qw_sim *s, const void *in, void *out, const Box &box, bool allow_fast) {
    StepArgs<R, 2 * DIM> a;
    fill_args<R, DIM>(s, in, out, box, a);
    const bool fast = allow_fast && s->coin_mode == QW_COIN_UNIFORM && !s->d_phases && !s->d_broken;
    if (fast && s->rbl && DIM == 2 && s->g.lattice == QW_NATURAL && (s->g.en & 1) == 0 && (a.n_lo & 1)) {
        a.n_lo -= 1; a.box_n += 1;      // even first column: lane pairs = generator groups (the extra site is a zero of the window)
    }
    // coin families on the vectorised path: per-walk matrices and / or site phases (natural lattice, no links)
    const bool fam = allow_fast && !fast && s->coin_mode != QW_COIN_PER_SITE && !s->d_broken && !s->rbl &&
                     s->g.lattice == QW_NATURAL;
    if (fam) {
        constexpr int UF = FusedShape<R, DIM>::U, BS = FusedShape<R, DIM>::BS;
        if (s->coin_mode == QW_COIN_UNIFORM) {         // uniform matrix + phases: keep the named coin's evaluation
            switch (s->coin_kind) {
                case COIN_HADAMARD: if (DIM == 1) return launch_scatter<R, DIM, COIN_HADAMARD, true, UF, false, BS, false, true>(s, a); break;
                case COIN_GROVER4:  if (DIM == 2) return launch_scatter<R, DIM, COIN_GROVER4, true, UF, false, BS, false, true>(s, a); break;
                case COIN_HXH4:     if (DIM == 2) return launch_scatter<R, DIM, COIN_HXH4, true, UF, false, BS, false, true>(s, a); break;
                case COIN_DFT4:     if (DIM == 2) return launch_scatter<R, DIM, COIN_DFT4, true, UF, false, BS, false, true>(s, a); break;
                default: break;
            }
        }
        return launch_scatter<R, DIM, COIN_GENERAL, true, UF, false, BS, false, true>(s, a);
    }
    if (fast) {
        if constexpr (DIM == 2) {
            if (s->g.lattice == QW_DIAGONAL)
                return s->rbl ? launch_fast_t<R, DIM, true, true>(s, a) : launch_fast_t<R, DIM, false, true>(s, a);
        }
        return s->rbl ? launch_fast_t<R, DIM, true, false>(s, a) : launch_fast_t<R, DIM, false, false>(s, a);
    }
    // the general kernel keeps the coin kind of the uniform matrix so that schedules agree bit for bit
    if (s->coin_mode == QW_COIN_UNIFORM) {
        switch (s->coin_kind) {
            case COIN_HADAMARD: if (DIM == 1) return launch_scatter<R, DIM, COIN_HADAMARD, false, 1>(s, a); break;
            case COIN_GROVER4:  if (DIM == 2) return launch_scatter<R, DIM, COIN_GROVER4, false, 1>(s, a); break;
            case COIN_HXH4:     if (DIM == 2) return launch_scatter<R, DIM, COIN_HXH4, false, 1>(s, a); break;
            case COIN_DFT4:     if (DIM == 2) return launch_scatter<R, DIM, COIN_DFT4, false, 1>(s, a); break;
            default: break;
        }
    }
    return launch_scatter<R, DIM, COIN_GENERAL, false, 1>(s, a);
}

int launch_step(qw_sim *s, const void *in, void *out, const Box &box, bool allow_fast) {
    if (s->dtype == QW_C128)
        return s->g.dim == 1 ? launch_step_t<double, 1>(s, in, out, box, allow_fast)
                             : launch_step_t<double, 2>(s, in, out, box, allow_fast);
    return s->g.dim == 1 ? launch_step_t<float, 1>(s, in, out, box, allow_fast)
                         : launch_step_t<float, 2>(s, in, out, box, allow_fast);
}

template <typename R, int DIM>
static int launch_inverse_t(qw_sim *s, const void *in, void *out) {
    StepArgs<R, 2 * DIM> a;
    Box full{0, s->g.em - 1, 0, s->g.en - 1};
    fill_args<R, DIM>(s, in, out, full, a);
    a.t = (unsigned)((unsigned long long)(s->t - 1) & 0xffffffffu);   // U(t-1)^dagger takes psi(t) back to psi(t-1)
    a.chunks_per_row = (int)((s->g.en + STEP_BLOCK - 1) / STEP_BLOCK);
    const long long blocks = s->g.batch * s->g.em * a.chunks_per_row;
    if (blocks > 0x7fffffffLL) return fail(QW_EUNSUPPORTED, "lattice too large for one launch");
    step_inverse_kernel<R, DIM><<<(unsigned)blocks, STEP_BLOCK, 0, s->stream>>>(a);
    QW_LAUNCH_CHECK(s, "step_inverse_kernel");
    return QW_OK;
}

int launch_step_inverse(qw_sim *s, const void *in, void *out) {
    if (s->dtype == QW_C128)
        return s->g.dim == 1 ? launch_inverse_t<double, 1>(s, in, out) : launch_inverse_t<double, 2>(s, in, out);
    return s->g.dim == 1 ? launch_inverse_t<float, 1>(s, in, out) : launch_inverse_t<float, 2>(s, in, out);
}

}  // namespace qw
