// qw_oracle.cpp — TEST INFRASTRUCTURE, NOT PRODUCT.
//
// Plain, slow, single-threaded, double-precision CPU implementation of the one-step
// evolution U = S (I (x) C) of a discrete-time coined quantum walk on Z^1 / Z^2
// (eq. 2, eq. 7), applied step by step.  The method is exact
// (psi(t) = U^t psi(0)), so this oracle IS the definition written out; the only
// freedom is rounding order.  It shares no code, header, table or helper with the CUDA
// path under paper_1003_3779_b200/csrc and neither side includes the other.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this library.  The product path never does.
//
// Conventions (readings of the paper; each is listed in DESIGN.md "Readings"):
//   state   psi[w][x][a]   walk w, site x, coin a; complex double, interleaved (re, im);
//           AoS layout [batch][site][coin]                         (PAPER.md:54-57 eq. 4, :73-78 eq. 6)
//   1D      coin 0 = R moves x -> x+1, coin 1 = L moves x -> x-1   ("|R> (+) |L>")
//   2D      coin c = 2j+k for the paper's |j,k>; site (m,n), index m*extent[1]+n;
//           natural lattice (eq. 8):  (m,n) -> (m + (-1)^j (1-d_jk), n + (-1)^j d_jk)
//             c0 -> (m, n+1)   c1 -> (m+1, n)   c2 -> (m-1, n)   c3 -> (m, n-1)
//           diagonal lattice (Fig. 1c; refs [8],[10]): (m,n) -> (m+(-1)^j, n+(-1)^k)
//   one step = coin first, then shift
//   periodic: indices modulo the extent
//   open:    a component whose link leaves the lattice (a broken link, RBL = 0 in
//            PAPER.md:94-101 eqs. 9-10) stays on its site with the opposite coin
//            (1D: 1-a; 2D: 3-c, i.e. (1-j,1-k)), no sign change.
//   broken links: an optional per-(walk, site, coin) byte mask marks the link
//            that component `a` of site x would leave through as broken; the component is
//            then treated exactly like the open-boundary case.  The caller supplies a
//            symmetric mask (both ends of a link agree); the oracle does not check that.
//
//   random broken links ("random broken links (termed RBL) technique", ref. [12]; eqs. 9-10):
//            qwo_step_rbl redraws the link states at EVERY step: each link of the lattice is broken
//            independently with probability p.  The paper names no generator; reading R27:
//            the state of a link is a pure function of (seed, walk, step, link) through the counter-based
//            generator Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11):
//              link    = (owner site, axis): the owner is the end from which the link points in the
//                        positive direction (dm > 0, or dm = 0 and dn > 0); axis = 0 for links along n
//                        (natural / 1D) or along (+1,+1) (diagonal), 1 for links along m or (+1,-1)
//              number  = owner index * dim + axis   (dim = links owned per site: 1 in 1D, 2 in 2D)
//              counter = (number / 4 low 32 bits, number / 4 high bits, step t, walk w), key = seed
//              broken  iff output word [number mod 4] < floor(p * 2^32)
//            (one generator call yields four independent words: it serves four consecutive links)
//            Links that leave an open lattice stay broken regardless.  Both ends of a link evaluate the
//            same function, so U(t) is unitary (pinned by the dense form).
//
// Parity status: every function here is pinned by tests/test_oracle_pins.py
// (hand/brute-force path sums, spectral closed form via FFT, Kronecker-product dense
// unitary, exact degenerate coins, invariants).  Nothing is "parity unpinned".

#include <cstdint>
#include <cstring>
#include <vector>

namespace {

struct cplx { double re, im; };

inline cplx cmul(cplx a, cplx b) { return { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re }; }
inline cplx cadd(cplx a, cplx b) { return { a.re + b.re, a.im + b.im }; }
inline cplx cconj(cplx a) { return { a.re, -a.im }; }

// Direction tables d_a = (dm, dn).  1D uses dn only.
const int DIR_1D[2][2]      = { {0, +1}, {0, -1} };
const int DIR_2D_NAT[4][2]  = { {0, +1}, {+1, 0}, {-1, 0}, {0, -1} };   // PAPER.md:88 eq. 8
const int DIR_2D_DIAG[4][2] = { {+1, +1}, {+1, -1}, {-1, +1}, {-1, -1} }; // PAPER.md:106 Fig. 1c

struct Lattice {
    int dim;            // 1 or 2
    int64_t em, en;     // extents: 1D -> em = 1, en = extent; 2D -> (em, en)
    int64_t sites;
    int cdim;           // 2 * dim
    int boundary;       // 0 periodic, 1 open (reflecting)
    const int (*dir)[2];
};

bool make_lattice(int dim, const int64_t* extents, int boundary, int lattice_kind, Lattice* L) {
    if (dim != 1 && dim != 2) return false;
    if (boundary != 0 && boundary != 1) return false;
    L->dim = dim;
    L->boundary = boundary;
    if (dim == 1) {
        if (extents[0] < 1) return false;
        L->em = 1; L->en = extents[0]; L->cdim = 2; L->dir = DIR_1D;
    } else {
        if (extents[0] < 1 || extents[1] < 1) return false;
        L->em = extents[0]; L->en = extents[1]; L->cdim = 4;
        L->dir = (lattice_kind == 1) ? DIR_2D_DIAG : DIR_2D_NAT;
    }
    L->sites = L->em * L->en;
    return true;
}

// Target of component a leaving site (m,n).  Returns false if the link leaves an open lattice.
inline bool target(const Lattice& L, int64_t m, int64_t n, int a, int64_t* tm, int64_t* tn) {
    int64_t y_m = m + L.dir[a][0];
    int64_t y_n = n + L.dir[a][1];
    if (L.boundary == 0) {
        y_m %= L.em; if (y_m < 0) y_m += L.em;
        y_n %= L.en; if (y_n < 0) y_n += L.en;
    } else {
        if (y_m < 0 || y_m >= L.em || y_n < 0 || y_n >= L.en) return false;
    }
    *tm = y_m; *tn = y_n;
    return true;
}

// Philox4x32-10, written from the published round function: two 32x32->64 multiplies by the constants
// M0, M1, the high halves XORed with the other counter words and the key, key bumped by the Weyl
// constants W0, W1 after every round; 10 rounds.
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = M0 * c0, p1 = M1 * c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Random broken links: is the link that component a of site (m,n) of walk w points along broken at step t?
// (header: "random broken links").  The link is assumed to stay inside the lattice (target() returned true
// with (tm,tn)).
inline bool rbl_broken(const Lattice& L, int64_t w, int64_t m, int64_t n, int a, int64_t tm, int64_t tn,
                       int64_t t, uint64_t thr, uint64_t seed) {
    const int dm = L.dir[a][0], dn = L.dir[a][1];
    const bool positive = dm > 0 || (dm == 0 && dn > 0);
    const int64_t owner = positive ? (m * L.en + n) : (tm * L.en + tn);
    int axis;
    if (dm != 0 && dn != 0) axis = (dm * dn > 0) ? 0 : 1;      // diagonal lattice
    else axis = (dm != 0) ? 1 : 0;                             // natural lattice / 1D
    // link number: the links of a walk are numbered owner * (links owned per site) + axis; one generator call serves
    // the four links 4g .. 4g+3 with its four output words (reading R27)
    const uint64_t link = (uint64_t)owner * (uint64_t)L.dim + (uint64_t)axis;
    const uint64_t group = link >> 2;
    const uint32_t ctr[4] = { (uint32_t)(group & 0xffffffffu), (uint32_t)(group >> 32),
                              (uint32_t)((uint64_t)t & 0xffffffffu), (uint32_t)((uint64_t)w & 0xffffffffu) };
    const uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    uint32_t out[4];
    philox4x32_10(ctr, key, out);
    return (uint64_t)out[link & 3u] < thr;
}

inline uint64_t rbl_threshold(double p) {       // floor(p * 2^32), p in [0, 1]
    return (uint64_t)(p * 4294967296.0);
}

inline const cplx* coin_at(const cplx* coin, int coin_mode, const Lattice& L, int64_t w, int64_t x) {
    const int64_t c2 = (int64_t)L.cdim * L.cdim;
    if (coin_mode == 0) return coin;
    if (coin_mode == 1) return coin + w * c2;
    return coin + (w * L.sites + x) * c2;
}

}  // namespace

extern "C" {

// n applications of U.  state: [batch][site][coin] complex, updated in place.
// coin: row-major cdim x cdim complex; coin_mode 0: one matrix, 1: batch matrices, 2: batch*sites.
// broken: nullptr, or [batch][site][coin] bytes (non-zero = the link component `coin` of that
//         site would cross is broken), constant over the n steps.
static int step_core(int dim, const int64_t* extents, int64_t batch, int boundary, int lattice_kind,
                     int coin_mode, const double* coin_, const uint8_t* broken, bool rbl, double p, uint64_t seed,
                     int64_t t0, double* state_, int64_t n) {
    const uint64_t thr = rbl ? rbl_threshold(p) : 0;
    Lattice L;
    if (!make_lattice(dim, extents, boundary, lattice_kind, &L) || batch < 1 || n < 0) return -1;
    const cplx* coin = reinterpret_cast<const cplx*>(coin_);
    cplx* state = reinterpret_cast<cplx*>(state_);
    const int cd = L.cdim;
    std::vector<cplx> phi((size_t)L.sites * cd), next((size_t)L.sites * cd);
    for (int64_t step = 0; step < n; ++step) {
        for (int64_t w = 0; w < batch; ++w) {
            cplx* psi = state + w * L.sites * cd;
            // 1. coin: phi[x][a] = sum_b C_x[a][b] psi[x][b]     (eq. 1)
            for (int64_t x = 0; x < L.sites; ++x) {
                const cplx* C = coin_at(coin, coin_mode, L, w, x);
                for (int a = 0; a < cd; ++a) {
                    cplx acc = {0.0, 0.0};
                    for (int b = 0; b < cd; ++b) acc = cadd(acc, cmul(C[a * cd + b], psi[x * cd + b]));
                    phi[x * cd + a] = acc;
                }
            }
            // 2. shift: psi'[x + d_a][a] = phi[x][a]               (PAPER.md:46 eq. 3, :88 eq. 8)
            //    broken / outward link: psi'[x][opposite(a)] = phi[x][a]   (eqs. 9-10)
            for (size_t i = 0; i < next.size(); ++i) next[i] = {0.0, 0.0};
            for (int64_t m = 0; m < L.em; ++m)
                for (int64_t nn = 0; nn < L.en; ++nn) {
                    const int64_t x = m * L.en + nn;
                    for (int a = 0; a < cd; ++a) {
                        int64_t tm, tn;
                        bool ok = target(L, m, nn, a, &tm, &tn);
                        if (ok && broken && broken[(w * L.sites + x) * cd + a]) ok = false;
                        if (ok && rbl && rbl_broken(L, w, m, nn, a, tm, tn, t0 + step, thr, seed)) ok = false;
                        if (ok) next[(tm * L.en + tn) * cd + a] = phi[x * cd + a];
                        else    next[x * cd + (cd - 1 - a)] = phi[x * cd + a];
                    }
                }
            // 3. psi <- psi'
            std::memcpy(psi, next.data(), next.size() * sizeof(cplx));
        }
    }
    return 0;
}

int qwo_step(int dim, const int64_t* extents, int64_t batch, int boundary, int lattice_kind,
             int coin_mode, const double* coin_, const uint8_t* broken, double* state_, int64_t n) {
    return step_core(dim, extents, batch, boundary, lattice_kind, coin_mode, coin_, broken, false, 0.0, 0, 0, state_, n);
}

// n applications of U(t), t = t0 .. t0+n-1, with the links redrawn at every step (header: "random broken links";
// PAPER.md:84, eqs. 9-10).  p in [0, 1].
int qwo_step_rbl(int dim, const int64_t* extents, int64_t batch, int boundary, int lattice_kind,
                 int coin_mode, const double* coin_, double p, uint64_t seed, int64_t t0, double* state_, int64_t n) {
    if (!(p >= 0.0 && p <= 1.0) || t0 < 0) return -1;
    return step_core(dim, extents, batch, boundary, lattice_kind, coin_mode, coin_, nullptr, true, p, seed, t0, state_, n);
}

// The link mask of step t as qwo_step's `broken` argument would take it: mask[w][x][a] = 1 iff the link component a
// of site x points along is broken at step t (links leaving an open lattice are not marked: they are always broken).
int qwo_rbl_mask(int dim, const int64_t* extents, int64_t batch, int boundary, int lattice_kind,
                 double p, uint64_t seed, int64_t t, uint8_t* mask) {
    Lattice L;
    if (!make_lattice(dim, extents, boundary, lattice_kind, &L) || batch < 1 || !(p >= 0.0 && p <= 1.0)) return -1;
    const uint64_t thr = rbl_threshold(p);
    for (int64_t w = 0; w < batch; ++w)
        for (int64_t m = 0; m < L.em; ++m)
            for (int64_t nn = 0; nn < L.en; ++nn)
                for (int a = 0; a < L.cdim; ++a) {
                    int64_t tm, tn;
                    const bool ok = target(L, m, nn, a, &tm, &tn);
                    mask[(w * L.sites + m * L.en + nn) * L.cdim + a] =
                        (ok && rbl_broken(L, w, m, nn, a, tm, tn, t, thr, seed)) ? 1 : 0;
                }
    return 0;
}

// The generator alone (known-answer pin).
void qwo_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

// n applications of U^dagger = (I (x) C^dagger) S^dagger (reversibility pin).
static int inverse_core(int dim, const int64_t* extents, int64_t batch, int boundary, int lattice_kind,
                        int coin_mode, const double* coin_, const uint8_t* broken, bool rbl, double p, uint64_t seed,
                        int64_t t0, double* state_, int64_t n) {
    const uint64_t thr = rbl ? rbl_threshold(p) : 0;
    Lattice L;
    if (!make_lattice(dim, extents, boundary, lattice_kind, &L) || batch < 1 || n < 0) return -1;
    const cplx* coin = reinterpret_cast<const cplx*>(coin_);
    cplx* state = reinterpret_cast<cplx*>(state_);
    const int cd = L.cdim;
    std::vector<cplx> phi((size_t)L.sites * cd);
    for (int64_t step = 0; step < n; ++step) {
        for (int64_t w = 0; w < batch; ++w) {
            cplx* psi = state + w * L.sites * cd;
            // undo the shift: phi[x][a] is read back from where the forward step wrote it
            for (int64_t m = 0; m < L.em; ++m)
                for (int64_t nn = 0; nn < L.en; ++nn) {
                    const int64_t x = m * L.en + nn;
                    for (int a = 0; a < cd; ++a) {
                        int64_t tm, tn;
                        bool ok = target(L, m, nn, a, &tm, &tn);
                        if (ok && broken && broken[(w * L.sites + x) * cd + a]) ok = false;
                        // inverse step number `step` undoes the forward step t0 - 1 - step
                        if (ok && rbl && rbl_broken(L, w, m, nn, a, tm, tn, t0 - 1 - step, thr, seed)) ok = false;
                        phi[x * cd + a] = ok ? psi[(tm * L.en + tn) * cd + a] : psi[x * cd + (cd - 1 - a)];
                    }
                }
            // undo the coin: psi[x][b] = sum_a conj(C_x[a][b]) phi[x][a]
            for (int64_t x = 0; x < L.sites; ++x) {
                const cplx* C = coin_at(coin, coin_mode, L, w, x);
                for (int b = 0; b < cd; ++b) {
                    cplx acc = {0.0, 0.0};
                    for (int a = 0; a < cd; ++a) acc = cadd(acc, cmul(cconj(C[a * cd + b]), phi[x * cd + a]));
                    psi[x * cd + b] = acc;
                }
            }
        }
    }
    return 0;
}

int qwo_step_inverse(int dim, const int64_t* extents, int64_t batch, int boundary, int lattice_kind,
                     int coin_mode, const double* coin_, const uint8_t* broken, double* state_, int64_t n) {
    return inverse_core(dim, extents, batch, boundary, lattice_kind, coin_mode, coin_, broken, false, 0.0, 0, 0, state_, n);
}

// Undo the n steps t0-1, t0-2, ..., t0-n of a random-broken-links walk (t0 = current time).
int qwo_step_inverse_rbl(int dim, const int64_t* extents, int64_t batch, int boundary, int lattice_kind,
                         int coin_mode, const double* coin_, double p, uint64_t seed, int64_t t0, double* state_, int64_t n) {
    if (!(p >= 0.0 && p <= 1.0) || t0 < n) return -1;
    return inverse_core(dim, extents, batch, boundary, lattice_kind, coin_mode, coin_, nullptr, true, p, seed, t0, state_, n);
}

// P[w][x] = sum_a |psi[w][x][a]|^2     (Figs. 3-4)
int qwo_probabilities(int dim, const int64_t* extents, int64_t batch, const double* state_, double* P) {
    Lattice L;
    if (!make_lattice(dim, extents, 0, 0, &L) || batch < 1) return -1;
    const cplx* state = reinterpret_cast<const cplx*>(state_);
    const int cd = L.cdim;
    for (int64_t i = 0; i < batch * L.sites; ++i) {
        double p = 0.0;
        for (int a = 0; a < cd; ++a) {
            const cplx z = state[i * cd + a];
            p += z.re * z.re + z.im * z.im;
        }
        P[i] = p;
    }
    return 0;
}

// Ensemble average over the batch: Pbar[x] = (1/batch) sum_w P[w][x], P as in qwo_probabilities; the
// averaged distribution of the random-broken-links model, every walk of
// the batch being one realisation of the links.  Plain definition: sum over the walks in order, then divide.
int qwo_probabilities_mean(int dim, const int64_t* extents, int64_t batch, const double* state_, double* Pbar) {
    Lattice L;
    if (!make_lattice(dim, extents, 0, 0, &L) || batch < 1) return -1;
    const cplx* state = reinterpret_cast<const cplx*>(state_);
    const int cd = L.cdim;
    for (int64_t x = 0; x < L.sites; ++x) {
        double sum = 0.0;
        for (int64_t w = 0; w < batch; ++w) {
            double p = 0.0;
            for (int a = 0; a < cd; ++a) {
                const cplx z = state[(w * L.sites + x) * cd + a];
                p += z.re * z.re + z.im * z.im;
            }
            sum += p;
        }
        Pbar[x] = sum / (double)batch;
    }
    return 0;
}

// Per walk: 1D {norm, mean, var}; 2D {norm, mean_m, mean_n, var_m, var_n, cov_mn}.
// Coordinates x_d = index_d - floor(extent_d / 2); moments divided by the computed norm;
// population variance.  Accumulated in long double so the oracle is the more accurate side.
int qwo_moments(int dim, const int64_t* extents, int64_t batch, const double* state_, double* out) {
    Lattice L;
    if (!make_lattice(dim, extents, 0, 0, &L) || batch < 1) return -1;
    const cplx* state = reinterpret_cast<const cplx*>(state_);
    const int cd = L.cdim;
    const int64_t cm = L.em / 2, cn = L.en / 2;
    for (int64_t w = 0; w < batch; ++w) {
        long double s0 = 0, sm = 0, sn = 0, smm = 0, snn = 0, smn = 0;
        for (int64_t m = 0; m < L.em; ++m)
            for (int64_t nn = 0; nn < L.en; ++nn) {
                const int64_t x = m * L.en + nn;
                long double p = 0;
                for (int a = 0; a < cd; ++a) {
                    const cplx z = state[(w * L.sites + x) * cd + a];
                    p += (long double)z.re * z.re + (long double)z.im * z.im;
                }
                const long double xm = (long double)(m - cm), xn = (long double)(nn - cn);
                s0 += p; sm += xm * p; sn += xn * p; smm += xm * xm * p; snn += xn * xn * p; smn += xm * xn * p;
            }
        if (dim == 1) {
            const long double mean = sn / s0;
            out[w * 3 + 0] = (double)s0;
            out[w * 3 + 1] = (double)mean;
            out[w * 3 + 2] = (double)(snn / s0 - mean * mean);
        } else {
            const long double mm = sm / s0, mn = sn / s0;
            out[w * 6 + 0] = (double)s0;
            out[w * 6 + 1] = (double)mm;
            out[w * 6 + 2] = (double)mn;
            out[w * 6 + 3] = (double)(smm / s0 - mm * mm);
            out[w * 6 + 4] = (double)(snn / s0 - mn * mn);
            out[w * 6 + 5] = (double)(smn / s0 - mm * mn);
        }
    }
    return 0;
}

// Dense matrix of U for one walk: column j = U e_j, obtained by one qwo_step on basis vector j.
// U is (sites*cdim)^2 complex, row-major.  Meant for <= 64 sites (brute-force pin P7).
int qwo_dense_unitary(int dim, const int64_t* extents, int boundary, int lattice_kind,
                      int coin_mode, const double* coin, const uint8_t* broken, double* U_) {
    Lattice L;
    if (!make_lattice(dim, extents, boundary, lattice_kind, &L)) return -1;
    const int64_t D = L.sites * L.cdim;
    cplx* U = reinterpret_cast<cplx*>(U_);
    std::vector<cplx> e((size_t)D);
    for (int64_t j = 0; j < D; ++j) {
        for (int64_t i = 0; i < D; ++i) e[i] = {0.0, 0.0};
        e[j] = {1.0, 0.0};
        int rc = qwo_step(dim, extents, 1, boundary, lattice_kind, coin_mode, coin, broken,
                          reinterpret_cast<double*>(e.data()), 1);
        if (rc) return rc;
        for (int64_t i = 0; i < D; ++i) U[i * D + j] = e[i];
    }
    return 0;
}

}  // extern "C"
