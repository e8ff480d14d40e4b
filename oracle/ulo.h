/* ulo.h -- ORACLE (test infrastructure, not the product).
 *
 * Plain, slow, single-threaded C++17 restatement of the hot path of
 * arXiv:1309.3859 (Amado, Cardoso, Bicudo): compact U(1) Wilson-action
 * heatbath + overrelaxation sweeps, slab-masked sub-updates and the
 * Luescher-Weisz multilevel estimator of <P^dagger P> and <P^dagger P O>.
 * All arithmetic is fp64 on link angles that are stored as fp32 (rounded on
 * store).  It shares no code with the CUDA path in paper_1309_3859_b200/.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.
 *
 * Citations: "P:<n>" = line n of /root/reference/PAPER.md; "S8(c)-O<k>" =
 * SURVEY.md section 8(c), item O<k>; "DESIGN R<k>" = reading k in DESIGN.md.
 *
 * Conventions: directions mu = 0 (time), 1,2,3 = x,y,z;
 * site index i = x1 + Ns*(x2 + Ns*(x3 + Ns*t)); parity (x1+x2+x3+t) mod 2;
 * canonical link array [mu][t][x3][x2][x1] (x1 fastest), fp32 radians.
 *
 * Every call returns 0 (ULO_OK) or a negative error code; nothing aborts.
 */
#ifndef ULO_H
#define ULO_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ulo_ctx ulo_ctx;
enum { ULO_OK = 0, ULO_EINVAL = -1, ULO_ENOMEM = -2, ULO_ESTATE = -4 };

/* lattice set-up.  ulo_create makes a hot start from `seed`. */
int ulo_create(ulo_ctx** h, int Ns, int Nt, double beta, uint64_t seed);
int ulo_destroy(ulo_ctx* h);
int ulo_init(ulo_ctx* h, int mode /*0 cold theta=0, 1 hot from seed (S8(c)-O4)*/);
int ulo_set_beta(ulo_ctx* h, double beta);
int ulo_set_links(ulo_ctx* h, const float* host /*[4][Nt][Ns][Ns][Ns]*/);
int ulo_get_links(ulo_ctx* h, float* host);
int ulo_get_counter(ulo_ctx* h, uint64_t* sweep_counter);
int ulo_set_counter(ulo_ctx* h, uint64_t sweep_counter);

/* updates: S8(c)-O1..O5 */
int ulo_sweep(ulo_ctx* h, int n_hb, int n_or);
int ulo_substep(ulo_ctx* h, int kind /*0 HB, 1 OR, 2 Metropolis*/, int parity, int mu, int slab_d /*0 = unmasked*/);
/* which algorithm the "n_hb" sweeps of ulo_sweep and of the sub-updates use: 0 = heatbath (default), 1 = one-hit
 * Metropolis with a uniform proposal of half-width delta in (0, pi] (DESIGN R21) */
int ulo_set_update_algorithm(ulo_ctx* h, int alg, double delta);
int ulo_set_subupdate(ulo_ctx* h, int n_hb, int n_or, int k_sweeps);
/* on = 1: the sums of T (row a7) use multihit temporal links for r >= 2; the TO sums keep the plain T */
int ulo_set_multihit(ulo_ctx* h, int on);

/* multilevel measurement: S8(c)-O6, O7; Alg. 1 */
int ulo_multilevel(ulo_ctx* h, int slab_thickness, int n_sub, int r_max,
                   const int* field_points /*[n_fp][3]*/, int n_fp);
int ulo_multilevel2(ulo_ctx* h, int d_in, int n_in, int d_out, int n_out, int r_max,
                    const int* field_points, int n_fp);
/* test hooks: open a single-level measurement, add the current configuration, close */
int ulo_measure_begin(ulo_ctx* h, int slab_thickness, int r_max, const int* field_points, int n_fp);
int ulo_accumulate(ulo_ctx* h);
int ulo_measure_end(ulo_ctx* h);
/* the same for two levels (S8(c)-O7; Alg. 1 lines 5, 16, 18): begin, then per outer iteration {ulo_accumulate of every
 * inner configuration, ulo_combine (Eqs. 32-33 on the inner averages, added to the outer sums)}, then end (outer
 * averages, slab product).  ulo_multilevel2 is exactly this sequence with its own sweeps in between. */
int ulo_measure2_begin(ulo_ctx* h, int d_in, int d_out, int r_max, const int* field_points, int n_fp);
int ulo_combine(ulo_ctx* h);
int ulo_measure2_end(ulo_ctx* h);

int ulo_plaquette(ulo_ctx* h, double* mean_cos /*[3]: all, time-like, space-like*/);
/* Polyakov-loop average <P> (Eqs. 15-16), out[2] = (Re, Im); multihit = 1: analytic multihit on every
 * temporal link, U_0 -> (I1(beta k)/I0(beta k)) e^{i alpha} */
int ulo_polyakov(ulo_ctx* h, int multihit, double* out);
int ulo_read_correlators(ulo_ctx* h, double* corr /*[r_max][2]*/,
                         double* field /*[r_max][n_fp][12][2]*/, double* vacuum /*[12]*/);
/* slab averages [T] of the last measurement (outer level for two-level):
 * out[((mu-1)*r_max + (r-1))*n_slab + s][xs][2], xs = x1 + Ns*(x2 + Ns*x3) */
int ulo_read_slab_averages(ulo_ctx* h, double* out);
/* slab averages [TO] of the last measurement (outer level for two-level):
 * out[(((mu-1)*r_max + (r-1))*n_slab + s)*n_fp + fp][ch][xs][2] */
int ulo_read_slab_field_averages(ulo_ctx* h, double* out);
const char* ulo_last_error(ulo_ctx* h);

/* ---- extra oracle-only entry points used by the pins in tests/ ---- */
/* Philox4x32-10, S8(c)-O4 */
void ulo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* staple sum S = k e^{i alpha} of link (site, mu), S8(c)-O1 */
int ulo_staple(ulo_ctx* h, int mu, long site, double* k, double* alpha);
/* one heatbath draw phi ~ exp(a cos phi) with the O3 sampler, counter words
 * (c0,c1,c2) and low byte c3low; returns the number of attempts used */
int ulo_heatbath_phi(double a, uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2,
                     uint32_t c3low, double* phi, int* attempts);
/* naive Polyakov-loop correlator straight from Eq. 15 and Eq. 23:
 * out[r-1] = (1/(3 Ns^3)) sum_x sum_mu conj(P(x)) P(x + r mu), r = 1..r_max; also <P> */
int ulo_polyakov_naive(ulo_ctx* h, int r_max, double* corr /*[r_max][2]*/, double* mean_P /*[2]*/);
/* accumulator bytes the paper's formula gives: 2*8*volume*area/step */
double ulo_paper_accumulator_bytes(int Ns, int Nt, int step);

#ifdef __cplusplus
}
#endif
#endif
