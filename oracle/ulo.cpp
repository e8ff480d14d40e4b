// ulo.cpp -- ORACLE (test infrastructure, not the product).  See ulo.h.
//
// Plain single-threaded C++17, fp64 arithmetic on fp32-stored angles, written
// in the paper's order and notation so it can be checked against the paper by
// eye.  No blocking, no fusion, no SIMD, no code shared with the CUDA path.
//
// Parity status: every function here is pinned by tests/test_oracle_*.py
// (closed forms, invariants, known-answer vectors, brute force) EXCEPT the
// paper's own ensemble values (sigma, widths, the 1e-15 signal of P:205), which
// need the paper's statistics: "parity unpinned" for those (context only).
#include "ulo.h"

#include <cmath>
#include <complex>
#include <cstring>
#include <string>
#include <vector>

typedef std::complex<double> cplx;
static const double PI = 3.14159265358979323846264338327950288;
static const double TWO_PI = 2.0 * PI;

struct ulo_ctx {
    int Ns = 0, Nt = 0;
    long Vs = 0, V = 0;            // Ns^3, Ns^3*Nt
    double beta = 0;
    uint64_t seed = 0, sweep = 0;  // sweep = count of HB sweeps issued (S8(c)-O4)
    std::vector<float> th;         // [4][V] canonical, fp32 radians
    int sub_hb = 1, sub_or = 3, sub_k = 1;  // sub-update recipe (DESIGN R5)
    int alg = 0;                   // 0 = heatbath (north star), 1 = Metropolis (DESIGN R21) for the "n_hb" sweeps
    double met_delta = PI;         // Metropolis proposal half-width (radians)
    int multihit = 0;              // 1: two-link operators at r >= 2 are built from multihit temporal links
    // open single-level measurement
    bool open = false;
    int d = 0, r_max = 0, n_fp = 0, n_slab = 0;
    long n_acc = 0;
    std::vector<int> fps;
    std::vector<cplx> A;           // [3][r_max][n_slab][Vs]                    (row a7)
    std::vector<cplx> B;           // [3][r_max][n_slab][n_fp][12][Vs]          (row a8)
    std::vector<double> vac_sum;   // [12]
    // last result
    bool have = false;
    int res_r_max = 0, res_n_fp = 0, res_n_slab = 0;
    std::vector<double> corr, field, vacuum;
    std::vector<cplx> slab_avg;    // [3][r_max][n_slab][Vs]
    std::vector<cplx> slab_field_avg;  // [3][r_max][n_slab][n_fp][12][Vs]
    // open two-level measurement (S8(c)-O7): outer sums and the number of outer iterations combined so far
    bool open2 = false;
    int d_out = 0, n_outer = 0;
    long n_comb = 0;
    std::vector<cplx> A4, B4;      // [3][r_max][n_outer][Vs], [3][r_max][n_outer][n_fp][12][Vs]
    std::vector<double> vac4;      // [12]
    std::string err;
};

// ---------------------------------------------------------------- indexing
static inline long site_of(const ulo_ctx* c, int x1, int x2, int x3, int t) {
    const long Ns = c->Ns;
    return x1 + Ns * (x2 + Ns * (x3 + Ns * (long)t));
}
static inline void coords_of(const ulo_ctx* c, long i, int x[4]) {  // x[0]=t, x[1..3]=x1..x3
    const long Ns = c->Ns;
    x[1] = (int)(i % Ns); i /= Ns;
    x[2] = (int)(i % Ns); i /= Ns;
    x[3] = (int)(i % Ns); i /= Ns;
    x[0] = (int)i;
}
static inline int extent(const ulo_ctx* c, int dir) { return dir == 0 ? c->Nt : c->Ns; }
// site i displaced by `delta` lattice units along `dir`, periodic
static long hop(const ulo_ctx* c, long i, int dir, int delta) {
    int x[4];
    coords_of(c, i, x);
    const int L = extent(c, dir);
    int v = (x[dir] + delta) % L;
    if (v < 0) v += L;
    x[dir] = v;
    return site_of(c, x[1], x[2], x[3], x[0]);
}
static inline int parity_of(const ulo_ctx* c, long i) {
    int x[4];
    coords_of(c, i, x);
    return (x[0] + x[1] + x[2] + x[3]) & 1;
}
static inline double TH(const ulo_ctx* c, int mu, long i) { return (double)c->th[(size_t)mu * c->V + i]; }

static inline double wrap(double v) { return v - TWO_PI * std::nearbyint(v / TWO_PI); }  // S8(c)-O2

// ---------------------------------------------------------------- Philox (S8(c)-O4)
extern "C" void ulo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = M0 * (uint64_t)c0;
        const uint64_t p1 = M1 * (uint64_t)c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
static inline double U_of(uint32_t w) { return (double)(2u * (w >> 9) + 1u) * (1.0 / 16777216.0); }  // (0,1), 23 bits

// ---------------------------------------------------------------- staple (S8(c)-O1, row a2)
// S = k e^{i alpha} = sum_{nu != mu} [ e^{-i sigma+} + e^{-i sigma-} ],
// so that the local weight of theta = theta_mu(x) is exp(beta k cos(theta - alpha)) (Eq. 6).
static cplx staple(const ulo_ctx* c, int mu, long x) {
    cplx S(0.0, 0.0);
    const long xpm = hop(c, x, mu, +1);
    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
        const long xpn = hop(c, x, nu, +1);
        const long xmn = hop(c, x, nu, -1);
        const long xpm_mn = hop(c, xpm, nu, -1);
        const double sp = TH(c, nu, xpm) - TH(c, mu, xpn) - TH(c, nu, x);
        const double sm = -TH(c, nu, xpm_mn) - TH(c, mu, xmn) + TH(c, nu, xmn);
        S += cplx(std::cos(sp), -std::sin(sp));
        S += cplx(std::cos(sm), -std::sin(sm));
    }
    return S;
}
static void k_alpha(const cplx& S, double* k, double* alpha) {
    *k = std::hypot(S.real(), S.imag());
    *alpha = (*k == 0.0) ? 0.0 : std::atan2(S.imag(), S.real());
}

// ---------------------------------------------------------------- heatbath (S8(c)-O3, DESIGN R2)
// Best-Fisher wrapped-Cauchy rejection for phi ~ exp(a cos phi) on (-pi, pi).
// Word-to-variate map (DESIGN R19, as revised in round 2): a Philox block holds four words and an attempt needs two
// uniforms and a sign, so attempt n takes block n >> 1 (counter word 3 = (block << 8) | c3low) and, of that block,
// the word pair (w[0], w[1]) when n is even, (w[2], w[3]) when n is odd: u1 = U(first), u2 = U(second), and the
// sign is bit 0 of the first word (U() reads bits 9..31 only, so the sign is independent of u1).
static double heatbath_phi(double a, const uint32_t key[2], uint32_t c0, uint32_t c1, uint32_t c2,
                           uint32_t c3low, int* attempts_out) {
    const double tau = 1.0 + std::sqrt(1.0 + 4.0 * a * a);
    const double s = tau + std::sqrt(2.0 * tau);
    const double rho = 2.0 * a / s;
    const double q = (1.0 - rho) / (1.0 + rho);
    const double ar = (1.0 + rho * rho) * s / 4.0;
    double phi = 0.0;
    int n = 0;
    uint32_t w[4] = {0, 0, 0, 0};
    for (; n < 64; ++n) {
        if ((n & 1) == 0) {
            const uint32_t ctr[4] = {c0, c1, c2, ((uint32_t)(n >> 1) << 8) | c3low};
            ulo_philox4x32_10(ctr, key, w);
        }
        const uint32_t wa = w[2 * (n & 1)], wb = w[2 * (n & 1) + 1];
        const double u1 = U_of(wa);
        const double u2 = U_of(wb);
        const double sgn = (wa & 1u) ? -1.0 : 1.0;
        const double T = q * std::tan(PI * u1 / 2.0);
        const double f = (1.0 - T * T) / (1.0 + T * T);
        const double cc = ar - a * f;
        phi = sgn * 2.0 * std::atan(T);
        if (u2 <= cc * std::exp(1.0 - cc)) { ++n; break; }
    }
    if (attempts_out) *attempts_out = n;  // number of attempts made (cap 64: the last proposal is kept)
    return phi;
}

static inline uint32_t c3_low(int tag, int parity, int mu) {
    return ((uint32_t)tag << 3) | ((uint32_t)parity << 2) | (uint32_t)mu;
}

// ---------------------------------------------------------------- updates (S8(c)-O2, O3, O5)
static inline bool frozen(const ulo_ctx* c, int mu, long x, int slab_d) {  // row a6
    if (slab_d <= 0 || mu == 0) return false;
    int xx[4];
    coords_of(c, x, xx);
    return (xx[0] % slab_d) == 0;
}
static void substep(ulo_ctx* c, int kind, int parity, int mu, int slab_d) {
    const uint32_t key[2] = {(uint32_t)(c->seed & 0xffffffffu), (uint32_t)(c->seed >> 32)};
    for (long x = 0; x < c->V; ++x) {
        if (parity_of(c, x) != parity) continue;
        if (frozen(c, mu, x, slab_d)) continue;
        double k, alpha;
        k_alpha(staple(c, mu, x), &k, &alpha);
        double theta_new;
        if (kind == 1) {
            theta_new = wrap(2.0 * alpha - TH(c, mu, x));                   // overrelaxation, O2
        } else if (kind == 2) {
            // Metropolis ("standard Metropolis algorithm"; DESIGN R21: the paper gives no proposal, so:
            // one hit, symmetric uniform proposal theta' = theta + delta (2 u1 - 1), accepted with probability
            // min(1, exp(-dS)) where -dS = beta k [cos(theta' - alpha) - cos(theta - alpha)] (Eq. 6).
            // Philox tag 3, attempt 0.  A rejected link keeps its stored value bit for bit.
            const uint32_t ctr[4] = {(uint32_t)x, (uint32_t)(c->sweep & 0xffffffffu), (uint32_t)(c->sweep >> 32), c3_low(3, parity, mu)};
            uint32_t w[4];
            ulo_philox4x32_10(ctr, key, w);
            const double u1 = U_of(w[0]), u2 = U_of(w[1]);
            const double theta = TH(c, mu, x);
            const double prop = theta + c->met_delta * (2.0 * u1 - 1.0);
            const double gain = c->beta * k * (std::cos(prop - alpha) - std::cos(theta - alpha));
            if (!(u2 <= std::exp(gain))) continue;
            theta_new = wrap(prop);
        } else {
            const double phi = heatbath_phi(c->beta * k, key, (uint32_t)x, (uint32_t)(c->sweep & 0xffffffffu),
                                            (uint32_t)(c->sweep >> 32), c3_low(0, parity, mu), nullptr);
            theta_new = wrap(alpha + phi);                                   // heatbath, O3
        }
        c->th[(size_t)mu * c->V + x] = (float)theta_new;                     // round to fp32 on store
    }
}
static void one_sweep(ulo_ctx* c, int kind, int slab_d) {  // O5: parity outer, direction inner
    for (int parity = 0; parity < 2; ++parity)
        for (int mu = 0; mu < 4; ++mu) substep(c, kind, parity, mu, slab_d);
    if (kind != 1) c->sweep += 1;                                            // heatbath and Metropolis sweeps consume the counter
}
static void compound(ulo_ctx* c, int n_hb, int n_or, int slab_d) {
    for (int i = 0; i < n_hb; ++i) one_sweep(c, c->alg == 1 ? 2 : 0, slab_d);   // the stochastic sweeps: heatbath or Metropolis
    for (int i = 0; i < n_or; ++i) one_sweep(c, 1, slab_d);
}

// ---------------------------------------------------------------- plaquettes
// theta_P(a,b)(y) = theta_a(y) + theta_b(y+a) - theta_a(y+b) - theta_b(y)
static double plaq_angle(const ulo_ctx* c, int a, int b, long y) {
    return TH(c, a, y) + TH(c, b, hop(c, y, a, +1)) - TH(c, a, hop(c, y, b, +1)) - TH(c, b, y);
}

// charge-aligned frame: nu = 1 + (mu mod 3), rho = 1 + ((mu+1) mod 3)
static inline void frame_of(int mu, int* nu, int* rho) { *nu = 1 + (mu % 3); *rho = 1 + ((mu + 1) % 3); }
// channel comp 0..5 -> plaquette orientation (a,b) in the frame of charge axis mu
static inline void comp_dirs(int mu, int comp, int* a, int* b) {
    int nu, rho;
    frame_of(mu, &nu, &rho);
    switch (comp) {
        case 0: *a = 0;   *b = mu;  break;   // E parallel
        case 1: *a = 0;   *b = nu;  break;   // E perp
        case 2: *a = 0;   *b = rho; break;   // E perp
        case 3: *a = nu;  *b = rho; break;   // B parallel
        case 4: *a = rho; *b = mu;  break;   // B perp
        default:*a = mu;  *b = nu;  break;   // B perp
    }
}
static inline double O_of(double thP, int kind) { return kind == 0 ? 1.0 - std::cos(thP) : std::sin(thP); }

// ---------------------------------------------------------------- measurement (S8(c)-O6; rows a7, a8, a10)
static inline size_t A_idx(const ulo_ctx* c, int mu, int r, int s, long xs) {
    return ((((size_t)(mu - 1) * c->r_max + (r - 1)) * c->n_slab + s) * c->Vs) + xs;
}
static inline size_t B_idx(const ulo_ctx* c, int mu, int r, int s, int fp, int ch, long xs) {
    return ((((((size_t)(mu - 1) * c->r_max + (r - 1)) * c->n_slab + s) * c->n_fp + fp) * 12 + ch) * c->Vs) + xs;
}
static int check_meas_args(ulo_ctx* c, int d, int r_max, const int* fps, int n_fp) {
    if (d < 1 || c->Nt % d != 0) { c->err = "Nt % slab_thickness != 0"; return ULO_EINVAL; }
    if (r_max < 1 || r_max > c->Ns / 2) { c->err = "r_max out of range [1, Ns/2]"; return ULO_EINVAL; }
    if (n_fp < 0 || (n_fp > 0 && !fps)) { c->err = "bad field points"; return ULO_EINVAL; }
    return ULO_OK;
}
static void open_measurement(ulo_ctx* c, int d, int r_max, const int* fps, int n_fp) {
    c->d = d; c->r_max = r_max; c->n_fp = n_fp; c->n_slab = c->Nt / d;
    c->fps.assign(fps, fps + 3 * (size_t)n_fp);
    c->A.assign((size_t)3 * r_max * c->n_slab * c->Vs, cplx(0, 0));
    c->B.assign((size_t)3 * r_max * c->n_slab * n_fp * 12 * c->Vs, cplx(0, 0));
    c->vac_sum.assign(12, 0.0);
    c->n_acc = 0;
    c->open = true;
}
// Ubar_0(x) = (I1(beta k)/I0(beta k)) e^{i alpha}, k e^{i alpha} the staple sum of the temporal link at site x
static cplx multihit_link(const ulo_ctx* c, long x) {
    double k, alpha;
    k_alpha(staple(c, 0, x), &k, &alpha);
    const double a = c->beta * k;
    const double ratio = a == 0.0 ? 0.0 : std::cyl_bessel_i(1.0, a) / std::cyl_bessel_i(0.0, a);
    return ratio * cplx(std::cos(alpha), std::sin(alpha));
}
// add the current configuration: A += T^(d), B += TO^(d)   (Eq. 25, Eq. 31 P:340 generalised to thickness d)
static void accumulate(ulo_ctx* c) {
    const int Ns = c->Ns;
    for (int s = 0; s < c->n_slab; ++s)
        for (int x3 = 0; x3 < Ns; ++x3)
            for (int x2 = 0; x2 < Ns; ++x2)
                for (int x1 = 0; x1 < Ns; ++x1) {
                    const long xs = x1 + (long)Ns * (x2 + (long)Ns * x3);
                    for (int mu = 1; mu <= 3; ++mu) {
                        int nu, rho;
                        frame_of(mu, &nu, &rho);
                        for (int r = 1; r <= c->r_max; ++r) {
                            // T^(d)(x,s,r mu) = prod_{t in slab} U0^dagger(x,t) U0(x + r mu, t)   (Eq. 22)
                            double phase = 0.0;
                            for (int t = s * c->d; t < (s + 1) * c->d; ++t) {
                                const long x = site_of(c, x1, x2, x3, t);
                                phase += TH(c, 0, hop(c, x, mu, r)) - TH(c, 0, x);
                            }
                            const cplx T2(std::cos(phase), std::sin(phase));
                            cplx TA = T2;
                            if (c->multihit && r >= 2) {
                                // analytic multihit: every temporal link of the two
                                // lines is replaced by its mean over its own local weight, Ubar = (I1/I0)(beta k) e^{i alpha};
                                // for r >= 2 no link of one line appears in the staple of a link of the other, and the
                                // links of one line never share a plaquette, so all 2 d replacements are independent
                                TA = cplx(1.0, 0.0);
                                for (int t = s * c->d; t < (s + 1) * c->d; ++t) {
                                    const long x = site_of(c, x1, x2, x3, t);
                                    TA *= std::conj(multihit_link(c, x)) * multihit_link(c, hop(c, x, mu, r));
                                }
                            }
                            c->A[A_idx(c, mu, r, s, xs)] += TA;
                            for (int fp = 0; fp < c->n_fp; ++fp) {
                                const int a = c->fps[3 * fp], b = c->fps[3 * fp + 1], cc = c->fps[3 * fp + 2];
                                for (int ch = 0; ch < 12; ++ch) {
                                    int pa, pb;
                                    comp_dirs(mu, ch / 2, &pa, &pb);
                                    double Osum = 0.0;
                                    for (int t = s * c->d; t < (s + 1) * c->d; ++t) {
                                        long y = site_of(c, x1, x2, x3, t);
                                        y = hop(c, y, mu, r / 2 + a);   // anchor: x + (floor(r/2)+a) mu + b nu + c rho  (DESIGN R10)
                                        y = hop(c, y, nu, b);
                                        y = hop(c, y, rho, cc);
                                        Osum += O_of(plaq_angle(c, pa, pb, y), ch % 2);
                                    }
                                    c->B[B_idx(c, mu, r, s, fp, ch, xs)] += T2 * Osum;
                                }
                            }
                        }
                    }
                }
    // vacuum <O_ch>: mean over all sites, all t, the three frames
    for (int ch = 0; ch < 12; ++ch) {
        double sum = 0.0;
        for (int mu = 1; mu <= 3; ++mu) {
            int pa, pb;
            comp_dirs(mu, ch / 2, &pa, &pb);
            for (long y = 0; y < c->V; ++y) sum += O_of(plaq_angle(c, pa, pb, y), ch % 2);
        }
        c->vac_sum[ch] += sum / (3.0 * (double)c->V);
    }
    c->n_acc += 1;
}
// C(r), G(r,fp,ch) from slab averages avT [3][r_max][n_slab][Vs], avTO [3][r_max][n_slab][n_fp][12][Vs]  (row a10)
static void reduce_result(ulo_ctx* c, const std::vector<cplx>& avT, const std::vector<cplx>& avTO,
                          int n_slab, const std::vector<double>& vac) {
    const int R = c->r_max, F = c->n_fp;
    c->corr.assign(2 * (size_t)R, 0.0);
    c->field.assign(2 * (size_t)R * F * 12, 0.0);
    for (int r = 1; r <= R; ++r) {
        cplx C(0, 0);
        std::vector<cplx> G((size_t)F * 12, cplx(0, 0));
        for (long xs = 0; xs < c->Vs; ++xs)
            for (int mu = 1; mu <= 3; ++mu) {
                auto Tat = [&](int s) { return avT[((((size_t)(mu - 1) * R + (r - 1)) * n_slab + s) * c->Vs) + xs]; };
                cplx prod(1, 0);
                for (int s = 0; s < n_slab; ++s) prod *= Tat(s);             // Eq. 26
                C += prod;
                for (int fp = 0; fp < F; ++fp)
                    for (int ch = 0; ch < 12; ++ch)
                        for (int s = 0; s < n_slab; ++s) {                    // Eq. 34
                            cplx term = avTO[((((((size_t)(mu - 1) * R + (r - 1)) * n_slab + s) * F + fp) * 12 + ch) * c->Vs) + xs];
                            for (int s2 = 0; s2 < n_slab; ++s2)
                                if (s2 != s) term *= Tat(s2);
                            G[(size_t)fp * 12 + ch] += term;
                        }
            }
        C /= 3.0 * (double)c->Vs;
        c->corr[2 * (r - 1)] = C.real();
        c->corr[2 * (r - 1) + 1] = C.imag();
        for (int fp = 0; fp < F; ++fp)
            for (int ch = 0; ch < 12; ++ch) {
                const cplx g = G[(size_t)fp * 12 + ch] / (3.0 * (double)c->Vs * (double)c->Nt);   // DESIGN R9
                const size_t o = 2 * ((((size_t)(r - 1)) * F + fp) * 12 + ch);
                c->field[o] = g.real();
                c->field[o + 1] = g.imag();
            }
    }
    c->vacuum = vac;
    c->slab_avg = avT;
    c->slab_field_avg = avTO;
    c->res_r_max = R; c->res_n_fp = F; c->res_n_slab = n_slab;
    c->have = true;
}
static void close_measurement(ulo_ctx* c) {
    const double inv = 1.0 / (double)c->n_acc;
    std::vector<cplx> avT(c->A), avTO(c->B);
    for (auto& z : avT) z *= inv;                                            // [.] = sum / n_sub
    for (auto& z : avTO) z *= inv;
    std::vector<double> vac(c->vac_sum);
    for (auto& v : vac) v *= inv;
    reduce_result(c, avT, avTO, c->n_slab, vac);
    c->open = false;
    c->A.clear(); c->A.shrink_to_fit();
    c->B.clear(); c->B.shrink_to_fit();
}

// ---------------------------------------------------------------- C ABI
extern "C" {

int ulo_create(ulo_ctx** h, int Ns, int Nt, double beta, uint64_t seed) {
    if (!h) return ULO_EINVAL;
    *h = nullptr;
    if (Ns < 2 || Nt < 2 || (Ns & 1) || (Nt & 1) || !(beta >= 0.0)) return ULO_EINVAL;
    ulo_ctx* c = new (std::nothrow) ulo_ctx;
    if (!c) return ULO_ENOMEM;
    c->Ns = Ns; c->Nt = Nt; c->Vs = (long)Ns * Ns * Ns; c->V = c->Vs * Nt;
    c->beta = beta; c->seed = seed; c->sweep = 0;
    try { c->th.assign((size_t)4 * c->V, 0.0f); } catch (...) { delete c; return ULO_ENOMEM; }
    *h = c;
    return ulo_init(c, 1);
}
int ulo_destroy(ulo_ctx* h) { delete h; return ULO_OK; }

int ulo_init(ulo_ctx* c, int mode) {
    if (!c || (mode != 0 && mode != 1)) return ULO_EINVAL;
    if (mode == 0) { std::fill(c->th.begin(), c->th.end(), 0.0f); return ULO_OK; }
    const uint32_t key[2] = {(uint32_t)(c->seed & 0xffffffffu), (uint32_t)(c->seed >> 32)};
    for (int mu = 0; mu < 4; ++mu)
        for (long x = 0; x < c->V; ++x) {
            const uint32_t ctr[4] = {(uint32_t)x, 0u, 0u, (1u << 3) | (uint32_t)mu};   // tag 1 = hot start
            uint32_t w[4];
            ulo_philox4x32_10(ctr, key, w);
            c->th[(size_t)mu * c->V + x] = (float)(TWO_PI * (double)w[0] * (1.0 / 4294967296.0) - PI);
        }
    return ULO_OK;
}
int ulo_set_beta(ulo_ctx* c, double beta) {
    if (!c || !(beta >= 0.0)) return ULO_EINVAL;
    c->beta = beta;
    return ULO_OK;
}
int ulo_set_links(ulo_ctx* c, const float* host) {
    if (!c || !host) return ULO_EINVAL;
    std::memcpy(c->th.data(), host, sizeof(float) * 4 * (size_t)c->V);
    return ULO_OK;
}
int ulo_get_links(ulo_ctx* c, float* host) {
    if (!c || !host) return ULO_EINVAL;
    std::memcpy(host, c->th.data(), sizeof(float) * 4 * (size_t)c->V);
    return ULO_OK;
}
int ulo_get_counter(ulo_ctx* c, uint64_t* v) { if (!c || !v) return ULO_EINVAL; *v = c->sweep; return ULO_OK; }
int ulo_set_counter(ulo_ctx* c, uint64_t v) { if (!c) return ULO_EINVAL; c->sweep = v; return ULO_OK; }

int ulo_sweep(ulo_ctx* c, int n_hb, int n_or) {
    if (!c || n_hb < 0 || n_or < 0) return ULO_EINVAL;
    compound(c, n_hb, n_or, 0);
    return ULO_OK;
}
int ulo_substep(ulo_ctx* c, int kind, int parity, int mu, int slab_d) {
    if (!c || kind < 0 || kind > 2 || (parity != 0 && parity != 1) || mu < 0 || mu > 3 || slab_d < 0) return ULO_EINVAL;
    if (slab_d > 0 && c->Nt % slab_d != 0) return ULO_EINVAL;
    substep(c, kind, parity, mu, slab_d);   // HB draws with the current counter and does not advance it
    return ULO_OK;
}
int ulo_set_update_algorithm(ulo_ctx* c, int alg, double delta) {
    if (!c || (alg != 0 && alg != 1) || (alg == 1 && !(delta > 0.0 && delta <= PI))) return ULO_EINVAL;
    c->alg = alg;
    if (alg == 1) c->met_delta = delta;
    return ULO_OK;
}
int ulo_set_multihit(ulo_ctx* c, int on) {
    if (!c || (on != 0 && on != 1)) return ULO_EINVAL;
    c->multihit = on;
    return ULO_OK;
}
int ulo_set_subupdate(ulo_ctx* c, int n_hb, int n_or, int k_sweeps) {
    if (!c || n_hb < 0 || n_or < 0 || k_sweeps < 1) return ULO_EINVAL;
    c->sub_hb = n_hb; c->sub_or = n_or; c->sub_k = k_sweeps;
    return ULO_OK;
}

int ulo_measure_begin(ulo_ctx* c, int d, int r_max, const int* fps, int n_fp) {
    if (!c) return ULO_EINVAL;
    int rc = check_meas_args(c, d, r_max, fps, n_fp);
    if (rc) return rc;
    try { open_measurement(c, d, r_max, fps, n_fp); } catch (...) { c->err = "accumulators do not fit"; return ULO_ENOMEM; }
    return ULO_OK;
}
int ulo_accumulate(ulo_ctx* c) {
    if (!c) return ULO_EINVAL;
    if (!c->open) { c->err = "no open measurement"; return ULO_ESTATE; }
    accumulate(c);
    return ULO_OK;
}
int ulo_measure_end(ulo_ctx* c) {
    if (!c) return ULO_EINVAL;
    if (!c->open || c->open2 || c->n_acc == 0) { c->err = "nothing accumulated (or a two-level measurement is open)"; return ULO_ESTATE; }
    close_measurement(c);
    return ULO_OK;
}

// single level, S8(c)-O6: sub-update j = k_sweeps masked compound sweeps, then measure; the starting
// configuration is not measured; n_sub = 0 measures the current configuration once.
int ulo_multilevel(ulo_ctx* c, int d, int n_sub, int r_max, const int* fps, int n_fp) {
    if (!c || n_sub < 0) return ULO_EINVAL;
    int rc = ulo_measure_begin(c, d, r_max, fps, n_fp);
    if (rc) return rc;
    if (n_sub == 0) accumulate(c);
    for (int j = 0; j < n_sub; ++j) {
        for (int k = 0; k < c->sub_k; ++k) compound(c, c->sub_hb, c->sub_or, d);
        accumulate(c);
    }
    close_measurement(c);
    return ULO_OK;
}

// two levels, S8(c)-O7 (Eq. 27, Eqs. 32-33 P:343-347 with the t+2 reading DESIGN R7, Alg. 1).
// The three steps below are Alg. 1 lines 5 (open the outer sums), 16 (combine the inner averages of one outer
// iteration into T^(4), TO^(4) and add them to the outer sums) and 18 (outer averages, slab product); they are also
// exported as test hooks so that a harness can feed configurations one by one (ulo_accumulate in between).
static int begin2(ulo_ctx* c, int d_in, int d_out, int r_max, const int* fps, int n_fp) {
    int rc = check_meas_args(c, d_in, r_max, fps, n_fp);
    if (rc) return rc;
    if (d_out < d_in || d_out % d_in != 0 || c->Nt % d_out != 0) { c->err = "need d_in | d_out | Nt"; return ULO_EINVAL; }
    c->d_out = d_out; c->n_outer = c->Nt / d_out; c->n_comb = 0;
    try {
        c->A4.assign((size_t)3 * r_max * c->n_outer * c->Vs, cplx(0, 0));
        c->B4.assign((size_t)3 * r_max * c->n_outer * n_fp * 12 * c->Vs, cplx(0, 0));
        open_measurement(c, d_in, r_max, fps, n_fp);                         // A2, B2 <- 0
    } catch (...) { c->err = "accumulators do not fit"; return ULO_ENOMEM; }
    c->vac4.assign(12, 0.0);
    c->open2 = true;
    return ULO_OK;
}
static void combine2(ulo_ctx* c) {
    const int m = c->d_out / c->d, n_outer = c->n_outer, R = c->r_max, F = c->n_fp;
    const double inv = 1.0 / (double)c->n_acc;                               // [.] = inner sum / n_in
    for (long xs = 0; xs < c->Vs; ++xs)
        for (int mu = 1; mu <= 3; ++mu)
            for (int r = 1; r <= R; ++r)
                for (int S = 0; S < n_outer; ++S) {
                    cplx t4(1, 0);
                    for (int i = 0; i < m; ++i) t4 *= c->A[A_idx(c, mu, r, S * m + i, xs)] * inv;          // Eq. 32
                    c->A4[((((size_t)(mu - 1) * R + (r - 1)) * n_outer + S) * c->Vs) + xs] += t4;
                    for (int fp = 0; fp < F; ++fp)
                        for (int ch = 0; ch < 12; ++ch) {
                            cplx to4(0, 0);
                            for (int i = 0; i < m; ++i) {                                                   // Eq. 33
                                cplx term = c->B[B_idx(c, mu, r, S * m + i, fp, ch, xs)] * inv;
                                for (int i2 = 0; i2 < m; ++i2)
                                    if (i2 != i) term *= c->A[A_idx(c, mu, r, S * m + i2, xs)] * inv;
                                to4 += term;
                            }
                            c->B4[((((((size_t)(mu - 1) * R + (r - 1)) * n_outer + S) * F + fp) * 12 + ch) * c->Vs) + xs] += to4;
                        }
                }
    for (int ch = 0; ch < 12; ++ch) c->vac4[ch] += c->vac_sum[ch] * inv;
    c->n_comb += 1;
    // the next outer iteration starts its inner sums from zero
    std::fill(c->A.begin(), c->A.end(), cplx(0, 0));
    std::fill(c->B.begin(), c->B.end(), cplx(0, 0));
    std::fill(c->vac_sum.begin(), c->vac_sum.end(), 0.0);
    c->n_acc = 0;
}
static void end2(ulo_ctx* c) {
    const double invo = 1.0 / (double)c->n_comb;                             // [.] = outer sum / n_out
    for (auto& z : c->A4) z *= invo;
    for (auto& z : c->B4) z *= invo;
    for (auto& v : c->vac4) v *= invo;
    reduce_result(c, c->A4, c->B4, c->n_outer, c->vac4);
    c->open = false; c->open2 = false;
    c->A.clear(); c->A.shrink_to_fit();
    c->B.clear(); c->B.shrink_to_fit();
    c->A4.clear(); c->A4.shrink_to_fit();
    c->B4.clear(); c->B4.shrink_to_fit();
}
int ulo_multilevel2(ulo_ctx* c, int d_in, int n_in, int d_out, int n_out, int r_max, const int* fps, int n_fp) {
    if (!c || n_in < 1 || n_out < 1) return ULO_EINVAL;
    int rc = begin2(c, d_in, d_out, r_max, fps, n_fp);
    if (rc) return rc;
    for (int J = 0; J < n_out; ++J) {
        for (int k = 0; k < c->sub_k; ++k) compound(c, c->sub_hb, c->sub_or, d_out);
        for (int j = 0; j < n_in; ++j) {
            for (int k = 0; k < c->sub_k; ++k) compound(c, c->sub_hb, c->sub_or, d_in);
            accumulate(c);
        }
        combine2(c);
    }
    end2(c);
    return ULO_OK;
}
int ulo_measure2_begin(ulo_ctx* c, int d_in, int d_out, int r_max, const int* fps, int n_fp) {
    if (!c) return ULO_EINVAL;
    return begin2(c, d_in, d_out, r_max, fps, n_fp);
}
int ulo_combine(ulo_ctx* c) {
    if (!c) return ULO_EINVAL;
    if (!c->open2 || c->n_acc == 0) { c->err = "no open two-level measurement with accumulated configurations"; return ULO_ESTATE; }
    combine2(c);
    return ULO_OK;
}
int ulo_measure2_end(ulo_ctx* c) {
    if (!c) return ULO_EINVAL;
    if (!c->open2 || c->n_comb == 0 || c->n_acc != 0) { c->err = "nothing combined, or configurations accumulated since the last combine"; return ULO_ESTATE; }
    end2(c);
    return ULO_OK;
}

int ulo_plaquette(ulo_ctx* c, double* out) {   // row a11, Eq. 6
    if (!c || !out) return ULO_EINVAL;
    double st = 0.0, ss = 0.0;
    for (long x = 0; x < c->V; ++x)
        for (int a = 0; a < 4; ++a)
            for (int b = a + 1; b < 4; ++b) {
                const double v = std::cos(plaq_angle(c, a, b, x));
                if (a == 0) st += v; else ss += v;
            }
    out[0] = (st + ss) / (6.0 * (double)c->V);
    out[1] = st / (3.0 * (double)c->V);
    out[2] = ss / (3.0 * (double)c->V);
    return ULO_OK;
}
int ulo_read_correlators(ulo_ctx* c, double* corr, double* field, double* vacuum) {
    if (!c) return ULO_EINVAL;
    if (!c->have) { c->err = "no measurement yet"; return ULO_ESTATE; }
    if (corr) std::memcpy(corr, c->corr.data(), sizeof(double) * c->corr.size());
    if (field && !c->field.empty()) std::memcpy(field, c->field.data(), sizeof(double) * c->field.size());
    if (vacuum) std::memcpy(vacuum, c->vacuum.data(), sizeof(double) * 12);
    return ULO_OK;
}
int ulo_read_slab_averages(ulo_ctx* c, double* out) {
    if (!c || !out) return ULO_EINVAL;
    if (!c->have) { c->err = "no measurement yet"; return ULO_ESTATE; }
    for (size_t i = 0; i < c->slab_avg.size(); ++i) { out[2 * i] = c->slab_avg[i].real(); out[2 * i + 1] = c->slab_avg[i].imag(); }
    return ULO_OK;
}
int ulo_read_slab_field_averages(ulo_ctx* c, double* out) {
    if (!c || !out) return ULO_EINVAL;
    if (!c->have) { c->err = "no measurement yet"; return ULO_ESTATE; }
    for (size_t i = 0; i < c->slab_field_avg.size(); ++i) { out[2 * i] = c->slab_field_avg[i].real(); out[2 * i + 1] = c->slab_field_avg[i].imag(); }
    return ULO_OK;
}
const char* ulo_last_error(ulo_ctx* c) { return c ? c->err.c_str() : "null handle"; }

int ulo_staple(ulo_ctx* c, int mu, long site, double* k, double* alpha) {
    if (!c || mu < 0 || mu > 3 || site < 0 || site >= c->V || !k || !alpha) return ULO_EINVAL;
    k_alpha(staple(c, mu, site), k, alpha);
    return ULO_OK;
}
int ulo_heatbath_phi(double a, uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3low,
                     double* phi, int* attempts) {
    if (!(a >= 0.0) || !phi) return ULO_EINVAL;
    const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
    *phi = heatbath_phi(a, key, c0, c1, c2, c3low & 0xffu, attempts);
    return ULO_OK;
}
// <P> = (1/Ns^3) sum_x prod_t U_0(x,t)  (Eqs. 15-16).  multihit = 1: every temporal link is replaced by
// its mean over the local weight exp(beta k cos(theta - alpha)) with all other links held fixed,
// U_0 -> (I1(beta k)/I0(beta k)) e^{i alpha} (analytic multihit, "when calculating the Polyakov loop average we
// also apply the analytical multihit integration technique"); k e^{i alpha} is the staple sum O1.  The links
// of one Polyakov line do not appear in each other's staples (Nt >= 2), so all Nt of them are replaced at once.
int ulo_polyakov(ulo_ctx* c, int multihit, double* out) {
    if (!c || !out || (multihit != 0 && multihit != 1)) return ULO_EINVAL;
    cplx mean(0, 0);
    for (long xs = 0; xs < c->Vs; ++xs) {
        cplx p(1, 0);
        for (int t = 0; t < c->Nt; ++t) {
            const long x = xs + c->Vs * t;
            if (!multihit) {
                const double th = TH(c, 0, x);
                p *= cplx(std::cos(th), std::sin(th));
            } else {
                double k, alpha;
                k_alpha(staple(c, 0, x), &k, &alpha);
                const double a = c->beta * k;
                const double ratio = a == 0.0 ? 0.0 : std::cyl_bessel_i(1.0, a) / std::cyl_bessel_i(0.0, a);
                p *= ratio * cplx(std::cos(alpha), std::sin(alpha));
            }
        }
        mean += p;
    }
    mean /= (double)c->Vs;
    out[0] = mean.real(); out[1] = mean.imag();
    return ULO_OK;
}
int ulo_polyakov_naive(ulo_ctx* c, int r_max, double* corr, double* mean_P) {
    if (!c || r_max < 0 || r_max > c->Ns / 2) return ULO_EINVAL;
    std::vector<cplx> P((size_t)c->Vs);
    cplx mean(0, 0);
    for (long xs = 0; xs < c->Vs; ++xs) {                    // Eq. 15
        cplx p(1, 0);
        for (int t = 0; t < c->Nt; ++t) {
            const double th = TH(c, 0, xs + c->Vs * t);
            p *= cplx(std::cos(th), std::sin(th));
        }
        P[(size_t)xs] = p;
        mean += p;
    }
    if (mean_P) { mean /= (double)c->Vs; mean_P[0] = mean.real(); mean_P[1] = mean.imag(); }   // Eq. 16
    for (int r = 1; r <= r_max && corr; ++r) {
        cplx C(0, 0);
        for (long xs = 0; xs < c->Vs; ++xs)
            for (int mu = 1; mu <= 3; ++mu) C += std::conj(P[(size_t)xs]) * P[(size_t)hop(c, xs, mu, r)];
        C /= 3.0 * (double)c->Vs;
        corr[2 * (r - 1)] = C.real();
        corr[2 * (r - 1) + 1] = C.imag();
    }
    return ULO_OK;
}
double ulo_paper_accumulator_bytes(int Ns, int Nt, int step) {
    const double volume = (double)Ns * Ns * Ns * Nt, area = (double)Ns * Ns;
    return 2.0 * 8.0 * volume * area / (double)step;
}

}  // extern "C"
