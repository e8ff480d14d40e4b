// ul_measure.cuh -- layout conversion, hot start, plaquette, and the multilevel estimator
// kernels.
//
// Accumulators are complex fp64 (double2) and every entry is owned by exactly one thread, so
// the sums are deterministic; lattice-wide sums use a fixed two-stage tree (block partials,
// then one block per output), never floating-point atomics (BJ kernel 4).
//
// Accumulator layouts (xs = x1 + Ns*(x2 + Ns*x3) fastest, so warps read-modify-write
// contiguous 512-byte runs):
//   A [mu-1][r-1][s][xs]             T^(d) sums          (row a7)
//   B [mu-1][r-1][s][fp][ch][xs]     TO^(d) sums         (row a8)
//   Th[s][xs]                        fixed-point slab sums of the temporal angles
//   Ot[o][kind][s][xs]               fp32 slab sums of O = 1-cos / sin of the 6 plaquette
//                                    orientations o: (0,1)(0,2)(0,3)(1,2)(1,3)(2,3)
#pragma once
#include "ul_math.cuh"

namespace ulk {

struct Geom {
    int Ns, Nh, Nt;
    long long Vs, V, Vh;
};

// address of theta_dir(t,x3,x2,x1) in the internal layout
__device__ __forceinline__ long long link_index(const Geom& g, int dir, int t, int x3, int x2, int x1) {
    const int par = (x1 + x2 + x3 + t) & 1;
    const long long row = ((long long)t * g.Ns + x3) * g.Ns + x2;
    return (long long)(dir * 2 + par) * g.Vh + row * g.Nh + (x1 >> 1);
}
__device__ __forceinline__ int wrapc(int v, int L) {          // v in [-L, 2L)
    v = (v >= L) ? v - L : v;
    return (v < 0) ? v + L : v;
}
__device__ __forceinline__ int modc(int v, int L) {           // any v
    v %= L;
    return (v < 0) ? v + L : v;
}

// ---------------------------------------------------------------- layout (row a1)
// canonical [mu][t][x3][x2][x1] <-> internal; pack = 1 (fp32 radians -> internal), 0 (internal -> fp32
// radians), 3 / 2 the same with raw int32 binary angles (bit copy).  On pack = 1, *bad is set if an angle
// is NaN or |theta| > 3.2.
__global__ void __launch_bounds__(256) k_repack(Geom g, int* __restrict__ internal, float* __restrict__ canonical,
                                                int pack, int* __restrict__ bad) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // over 4V canonical elements
    if (i >= 4 * g.V) return;
    const int mu = (int)(i / g.V);
    long long s = i - (long long)mu * g.V;
    const int x1 = (int)(s % g.Ns); s /= g.Ns;
    const int x2 = (int)(s % g.Ns); s /= g.Ns;
    const int x3 = (int)(s % g.Ns); s /= g.Ns;
    const int t = (int)s;
    const long long j = link_index(g, mu, t, x3, x2, x1);
    if (pack == 1) {
        const float v = canonical[i];
        if (!(fabsf(v) <= 3.2f)) *bad = 1;
        internal[j] = ulm::rad_to_bt(v);              // nearest binary angle (fp64 scaling)
    } else if (pack == 0) {
        canonical[i] = ulm::bt_to_rad(internal[j]);
    } else if (pack == 3) {                           // raw binary angles in canonical order (exact checkpoint)
        internal[j] = __float_as_int(canonical[i]);
    } else {
        canonical[i] = __int_as_float(internal[j]);
    }
}

// hot start (S8(c)-O4): theta = fp32(2 pi w0 2^-32 - pi), ctr = (site, 0, 0, (1<<3)|mu)
__global__ void __launch_bounds__(256) k_hot_start(Geom g, int* __restrict__ internal, uint32_t key0, uint32_t key1) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 4 * g.V) return;
    const int mu = (int)(i / g.V);
    long long s = i - (long long)mu * g.V;
    const uint32_t site = (uint32_t)s;
    const int x1 = (int)(s % g.Ns); s /= g.Ns;
    const int x2 = (int)(s % g.Ns); s /= g.Ns;
    const int x3 = (int)(s % g.Ns); s /= g.Ns;
    const int t = (int)s;
    uint32_t w[4];
    ulm::philox4x32_10(site, 0u, 0u, (1u << 3) | (uint32_t)mu, key0, key1, w);
    const double th = 6.28318530717958647692 * (double)w[0] * (1.0 / 4294967296.0) - 3.14159265358979323846;
    internal[link_index(g, mu, t, x3, x2, x1)] = ulm::rad_to_bt((float)th);
}

__global__ void k_philox_test(const uint32_t* __restrict__ ctr, const uint32_t* __restrict__ key, uint32_t* __restrict__ out, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t w[4];
    ulm::philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1], w);
    out[4 * i] = w[0]; out[4 * i + 1] = w[1]; out[4 * i + 2] = w[2]; out[4 * i + 3] = w[3];
}

// ---------------------------------------------------------------- fp64 block reduction (BJ kernel 4)
// Sums N doubles per thread over the block in a fixed order: warp shuffles, then warp 0 over
// the per-warp partials.  Result valid in thread 0.
template <int N>
__device__ __forceinline__ void block_sum(double v[N], double* smem /* [N][32] */) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int k = 0; k < N; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
        if (lane == 0) smem[k * 32 + wid] = v[k];
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int k = 0; k < N; ++k) {
            double x = (lane < nw) ? smem[k * 32 + lane] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
            v[k] = x;
        }
    }
    __syncthreads();
}

// out[k] (+)= sum_b partial[k*nblk + b], one block per k, fixed order
__global__ void __launch_bounds__(256) k_sum_partials(const double* __restrict__ partial, int nblk, double* __restrict__ out,
                                                      double scale, int accumulate) {
    __shared__ double sm[32];
    const int k = blockIdx.x;
    double v[1] = {0.0};
    for (int b = threadIdx.x; b < nblk; b += blockDim.x) v[0] += partial[(long long)k * nblk + b];
    block_sum<1>(v, sm);
    if (threadIdx.x == 0) out[k] = (accumulate ? out[k] : 0.0) + v[0] * scale;
}

// ---------------------------------------------------------------- plaquette angles
// theta_P(a,b)(x) = theta_a(x) + theta_b(x+a) - theta_a(x+b) - theta_b(x) as binary angles (wrapping adds:
// exact mod 2 pi) for the six orientations (0,1)(0,2)(0,3)(1,2)(1,3)(2,3) of site x; th0 = theta_0(x).
// 16 loads: the four links at x and the three transverse links at each of the four forward neighbours,
// addressed by 32-bit element offsets (4V < 2^31 is checked by ul_create).
__device__ __forceinline__ void site_plaquettes(const Geom& g, const int* __restrict__ th, const int x[4], int pl[6], int& th0) {
    const int Ns = g.Ns, Nh = g.Nh, Vh = (int)g.Vh;
    const int par = (x[0] + x[1] + x[2] + x[3]) & 1;
    const int row = (x[0] * Ns + x[3]) * Ns + x[2];
    const int e = row * Nh + (x[1] >> 1);
    int en[4];                                                     // element offsets of the sites x + b (parity 1 - par)
    en[0] = e + ((x[0] + 1 == g.Nt) ? -(g.Nt - 1) : 1) * Ns * Ns * Nh;
    en[1] = row * Nh + (((x[1] + 1 == Ns) ? 0 : x[1] + 1) >> 1);
    en[2] = e + ((x[2] + 1 == Ns) ? -(Ns - 1) : 1) * Nh;
    en[3] = e + ((x[3] + 1 == Ns) ? -(Ns - 1) : 1) * Ns * Nh;
    unsigned own[4], nb[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a) own[a] = (unsigned)__ldg(th + (2 * a + par) * Vh + e);
#pragma unroll
    for (int b = 0; b < 4; ++b)
#pragma unroll
        for (int a = 0; a < 4; ++a)
            if (a != b) nb[b][a] = (unsigned)__ldg(th + (2 * a + 1 - par) * Vh + en[b]);   // theta_a(x + b)
    int o = 0;
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = a + 1; b < 4; ++b) pl[o++] = (int)(own[a] + nb[a][b] - nb[b][a] - own[b]);
    th0 = (int)own[0];
}

// row a11: partial[0*nblk + b] = sum of cos over time-like plaquettes, [1*nblk + b] space-like
// Grid (ceil(Ns^2/256), rows): a thread keeps its (x1, x2) and walks over the (t, x3) rows, so the only
// divisions are one per thread and one per row (all 32-bit).
__global__ void __launch_bounds__(256) k_plaquette(Geom g, const int* __restrict__ th, double* __restrict__ partial) {
    __shared__ double sm[2 * 32];
    const unsigned Ns = (unsigned)g.Ns;
    const unsigned i2 = blockIdx.x * blockDim.x + threadIdx.x;
    const bool in = i2 < Ns * Ns;
    int x[4];
    x[2] = (int)(i2 / Ns);
    x[1] = (int)(i2 - (unsigned)x[2] * Ns);
    double v[2] = {0.0, 0.0};
    for (unsigned row = blockIdx.y; row < (unsigned)g.Nt * Ns; row += gridDim.y) {
        x[0] = (int)(row / Ns);
        x[3] = (int)(row - (unsigned)x[0] * Ns);
        if (!in) continue;
        int pl[6], th0;
        site_plaquettes(g, th, x, pl, th0);
        float ct = 0.0f, cs = 0.0f;
#pragma unroll
        for (int o = 0; o < 6; ++o) {
            float c, sn;
            ulm::sincos_bt(pl[o], c, sn);
            if (o < 3) ct += c; else cs += c;
        }
        v[0] += (double)ct;
        v[1] += (double)cs;
    }
    block_sum<2>(v, sm);
    const unsigned nblk = gridDim.x * gridDim.y, blk = blockIdx.y * gridDim.x + blockIdx.x;
    if (threadIdx.x == 0) { partial[blk] = v[0]; partial[nblk + blk] = v[1]; }
}

// ---------------------------------------------------------------- Polyakov-loop average (next row S8(f) rank 1)
// I1(a)/I0(a) in fp64 by the backward recurrence R_{n-1} = 1 / (2n/a + R_n), R_n = I_{n+1}/I_n, from R_N = 0 at
// N = a + 40 (each step contracts the error by R^2 < 0.4, so the start value is forgotten to 1e-18).
__device__ __forceinline__ double bessel_ratio_i1_i0(double a) {
    if (!(a > 1e-300)) return 0.0;
    const double two_over_a = 2.0 / a;
    double R = 0.0;
    for (int n = (int)a + 40; n >= 1; --n) R = 1.0 / ((double)n * two_over_a + R);
    return R;
}

// partial[b], partial[nblk + b] = block sums of Re, Im of P(x) = prod_t U_0(x,t) (Eq. 15) over the spatial sites;
// multihit = 1: U_0 -> (I1(beta k)/I0(beta k)) e^{i alpha} = (I1/I0)(beta k) S/k with the staple sum S = k e^{i alpha}
// (P:209), everything in fp64 on exact integer phase sums.  One thread per spatial site, grid-stride.
__global__ void __launch_bounds__(256) k_polyakov(Geom g, const int* __restrict__ th, double beta, int multihit,
                                                  double* __restrict__ partial) {
    __shared__ double sm[2 * 32];
    const int Ns = g.Ns, Nt = g.Nt;
    double v[2] = {0.0, 0.0};
    for (int xs = blockIdx.x * blockDim.x + threadIdx.x; xs < (int)g.Vs; xs += gridDim.x * blockDim.x) {
        int x[4];
        x[1] = xs % Ns;
        x[2] = (xs / Ns) % Ns;
        x[3] = xs / (Ns * Ns);
        double pr = 1.0, pi = 0.0;
        unsigned phase = 0u;
        for (int t = 0; t < Nt; ++t) {
            if (!multihit) {
                phase += (unsigned)__ldg(th + link_index(g, 0, t, x[3], x[2], x[1]));
                continue;
            }
            const int tp = (t + 1 == Nt) ? 0 : t + 1;
            double Sx = 0.0, Sy = 0.0;
#pragma unroll
            for (int nu = 1; nu <= 3; ++nu) {
                int yp[4] = {t, x[1], x[2], x[3]}, ym[4] = {t, x[1], x[2], x[3]};
                yp[nu] = (x[nu] + 1 == Ns) ? 0 : x[nu] + 1;
                ym[nu] = (x[nu] == 0) ? Ns - 1 : x[nu] - 1;
                // -sigma+ = th_nu(x) + th_0(x+nu) - th_nu(x+t);  -sigma- = th_nu(x+t-nu) + th_0(x-nu) - th_nu(x-nu)
                const unsigned sp = (unsigned)__ldg(th + link_index(g, nu, t, x[3], x[2], x[1]))
                                  + (unsigned)__ldg(th + link_index(g, 0, t, yp[3], yp[2], yp[1]))
                                  - (unsigned)__ldg(th + link_index(g, nu, tp, x[3], x[2], x[1]));
                const unsigned sn = (unsigned)__ldg(th + link_index(g, nu, tp, ym[3], ym[2], ym[1]))
                                  + (unsigned)__ldg(th + link_index(g, 0, t, ym[3], ym[2], ym[1]))
                                  - (unsigned)__ldg(th + link_index(g, nu, t, ym[3], ym[2], ym[1]));
                double c, s;
                ulm::sincos_bt_f64((int)sp, c, s); Sx += c; Sy += s;
                ulm::sincos_bt_f64((int)sn, c, s); Sx += c; Sy += s;
            }
            const double k = sqrt(Sx * Sx + Sy * Sy);
            const double f = k > 0.0 ? bessel_ratio_i1_i0(beta * k) / k : 0.0;             // (I1/I0) e^{i alpha} = f S
            const double ur = f * Sx, ui = f * Sy;
            const double nr = pr * ur - pi * ui;
            pi = pr * ui + pi * ur;
            pr = nr;
        }
        if (!multihit) ulm::sincos_bt_f64((int)phase, pr, pi);
        v[0] += pr;
        v[1] += pi;
    }
    block_sum<2>(v, sm);
    if (threadIdx.x == 0) { partial[blockIdx.x] = v[0]; partial[gridDim.x + blockIdx.x] = v[1]; }
}

// ---------------------------------------------------------------- per-configuration slab tables
// U[s][xs]  = exp(i sum_{t in slab s} theta_0(xs,t)) in fp64: the angle sum is a wrapping integer add
//             (exact mod 2 pi), reduced in integers and expanded in fp64 (sincos_bt_f64), so U is good to 1 ulp and
//             every T^(d)(x,s,r mu) = U(x + r mu) conj(U(x)) (Eqs. 22, 25) is one fp64 complex product.
// Ot[o][kind][s][xs] = sum_{t in slab s} O(theta_P(o)(xs,t)),  O = 1 - cos (kind 0), sin (kind 1); stored
//             only when field points are measured (Ot != nullptr).
// partial[col*nblk + b] = block partial of the column sums of O (vacuum expectation values).
// Grid (ceil(Ns^2/256), rows): a thread keeps its (x1, x2) and walks over the (s, x3) rows.
struct TableArgs {
    Geom g;
    const int* th;
    int d, n_slab;
    double2* U;
    double2* Um;          // multihit table (nullptr: off): prod_t Ubar_0(xs,t), Ubar = (I1/I0)(beta k) e^{i alpha}
    float beta;
    float* Ot;
    double* partial;
    int row0, n_rows;     // rows (s, x3) = s * Ns + x3 handled by this launch: [row0, row0 + n_rows)  (a range of slabs)
};

// I1(a)/I0(a) in fp32 by the backward recurrence R_{n-1} = 1/(2n/a + R_n) from R_N = 0, N = a + 20 (the start value is
// forgotten to 1e-8: every step contracts the error by R^2 < 0.4); MUFU.RCP per step, ~2e-7 relative
__device__ __forceinline__ float bessel_ratio_i1_i0_f32(float a) {
    if (!(a > 1e-30f)) return 0.0f;
    const float two_over_a = 2.0f * ulm::mufu_rcp(a);
    float R = 0.0f;
    for (int n = min((int)a, 1000) + 20; n >= 1; --n) R = ulm::mufu_rcp(fmaf((float)n, two_over_a, R));
    return R;
}

__global__ void __launch_bounds__(256) k_slab_tables(const TableArgs P) {
    __shared__ double sm[12 * 32];
    const Geom& g = P.g;
    const long long n = (long long)P.n_slab * g.Vs;
    const unsigned Ns = (unsigned)g.Ns;
    const unsigned i2 = blockIdx.x * blockDim.x + threadIdx.x;                 // (x1, x2) of this thread
    const bool in = i2 < Ns * Ns;
    int x[4];
    x[2] = (int)(i2 / Ns);
    x[1] = (int)(i2 - (unsigned)x[2] * Ns);
    float vf[12];                                   // per-thread column sums: a few terms of magnitude <= 2 each, then fp64
#pragma unroll
    for (int o = 0; o < 12; ++o) vf[o] = 0.0f;
    for (unsigned row = (unsigned)P.row0 + blockIdx.y; row < (unsigned)(P.row0 + P.n_rows); row += gridDim.y) {   // rows (s, x3): 32-bit divisions only
        const int s = (int)(row / Ns);
        x[3] = (int)(row - (unsigned)s * Ns);
        if (!in) continue;
        const long long idx = (long long)row * (Ns * Ns) + i2;
        unsigned acc = 0u;
        double mhr = 1.0, mhi = 0.0;                              // running product of the multihit factors f S' over the slab
        float o_c[6], o_s[6];
#pragma unroll
        for (int o = 0; o < 6; ++o) { o_c[o] = 0.0f; o_s[o] = 0.0f; }
        for (int t = s * P.d; t < (s + 1) * P.d; ++t) {
            x[0] = t;
            int pl[6], th0;
            site_plaquettes(g, P.th, x, pl, th0);
            acc += (unsigned)th0;
            float Sx = 0.0f, Sy = 0.0f;                           // S' = sum_i [e^{-i P_i} + e^{+i Q_i}]: the staple sum of theta_0(x,t)
#pragma unroll                                                    // is e^{i theta_0} S', P_i = theta_P(0,i)(x), Q_i = theta_P(0,i)(x - i)
            for (int o = 0; o < 6; ++o) {
                float c, sn;
                ulm::sincos_bt(pl[o], c, sn);
                o_c[o] += 1.0f - c;
                o_s[o] += sn;
                if (o < 3) { Sx += c; Sy -= sn; }
            }
            if (P.Um) {
                const int tp = (t + 1 == g.Nt) ? 0 : t + 1;
#pragma unroll
                for (int i = 1; i <= 3; ++i) {
                    int y[4] = {t, x[1], x[2], x[3]};
                    y[i] = (x[i] == 0) ? (int)Ns - 1 : x[i] - 1;
                    const unsigned q = (unsigned)__ldg(P.th + link_index(g, 0, t, y[3], y[2], y[1]))
                                     + (unsigned)__ldg(P.th + link_index(g, i, tp, y[3], y[2], y[1]))
                                     - (unsigned)th0 - (unsigned)__ldg(P.th + link_index(g, i, t, y[3], y[2], y[1]));
                    float c, sn;
                    ulm::sincos_bt((int)q, c, sn);
                    Sx += c; Sy += sn;
                }
                const float k2 = fmaf(Sx, Sx, Sy * Sy);
                const float k = ulm::mufu_sqrt(k2);
                const float f = k2 > 0.0f ? bessel_ratio_i1_i0_f32(P.beta * k) * ulm::mufu_rcp(k) : 0.0f;   // (I1/I0) e^{i alpha} = f e^{i theta_0} S'
                const double fr = (double)(f * Sx), fi = (double)(f * Sy);
                const double nr = mhr * fr - mhi * fi;
                mhi = mhr * fi + mhi * fr;
                mhr = nr;
            }
        }
        double us, uc;
        ulm::sincos_bt_f64((int)acc, uc, us);
        if (P.U) P.U[idx] = make_double2(uc, us);
        if (P.Um) P.Um[idx] = make_double2(uc * mhr - us * mhi, uc * mhi + us * mhr);
#pragma unroll
        for (int o = 0; o < 6; ++o) {
            if (P.Ot) {
                P.Ot[(long long)(2 * o) * n + idx] = o_c[o];
                P.Ot[(long long)(2 * o + 1) * n + idx] = o_s[o];
            }
            vf[2 * o] += o_c[o];
            vf[2 * o + 1] += o_s[o];
        }
    }
    double v[12];
#pragma unroll
    for (int o = 0; o < 12; ++o) v[o] = (double)vf[o];
    block_sum<12>(v, sm);
    if (threadIdx.x == 0) {
        const unsigned nblk = gridDim.x * gridDim.y, blk = blockIdx.y * gridDim.x + blockIdx.x;
#pragma unroll
        for (int o = 0; o < 12; ++o) P.partial[(long long)o * nblk + blk] = v[o];
    }
}

// The U table alone (no field points, no multihit: nothing needs the plaquettes): one thread per (row, h) = the two
// sites x1 = 2h, 2h + 1 of a row (t, x3, x2), whose temporal links sit at the same offset of the two parity arrays;
// reads V * 4 B, writes n_slab * Vs * 16 B, both coalesced (S8(d): the algorithmic traffic of row a7's table).
__global__ void __launch_bounds__(256) k_slab_tables_u(const TableArgs P) {
    const Geom& g = P.g;
    const int Ns = g.Ns, Nh = g.Nh;
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;                   // over (s - s0, x3, x2, h): < V/2 < 2^30, 32-bit divisions
    const unsigned total = (unsigned)P.n_rows * Ns * Nh;
    if (i >= total) return;
    const unsigned rr = i / (unsigned)Nh;                                       // (s - s0, x3, x2)
    const int h = (int)(i - rr * Nh);
    const unsigned rq = rr / (unsigned)Ns;
    const int x2 = (int)(rr - rq * Ns);
    const int row = P.row0 + (int)rq;                                           // s * Ns + x3
    const int s = row / Ns, x3 = row - s * Ns;
    unsigned acc0 = 0u, acc1 = 0u;                                              // parity-0 / parity-1 array element
    for (int t = s * P.d; t < (s + 1) * P.d; ++t) {
        const long long e = (((long long)t * Ns + x3) * Ns + x2) * Nh + h;
        // the site of parity par in this row pair is x1 = 2h + ((par + x2 + x3 + t) & 1): over a slab the two arrays swap
        // roles with t, so add each element to the sum of the x1 it belongs to
        const unsigned a = (unsigned)__ldg(P.th + e), b = (unsigned)__ldg(P.th + g.Vh + e);
        if ((x2 + x3 + t) & 1) { acc0 += b; acc1 += a; } else { acc0 += a; acc1 += b; }   // acc0: x1 = 2h, acc1: x1 = 2h + 1
    }
    double c0, s0, c1, s1;
    ulm::sincos_bt_f64((int)acc0, c0, s0);
    ulm::sincos_bt_f64((int)acc1, c1, s1);
    double2* out = P.U + (long long)row * (Ns * Ns) + (long long)x2 * Ns + 2 * h;
    out[0] = make_double2(c0, s0);                                               // the accumulation kernel re-reads U 6 r_max times:
    out[1] = make_double2(c1, s1);                                               // keep it in L2
}

// plaquette orientation (a,b) -> table column o and sign of the sin channel (theta_P(b,a) = -theta_P(a,b))
__device__ __forceinline__ void orient_of(int a, int b, int& o, float& sgn) {
    sgn = 1.0f;
    if (a > b) { const int c = a; a = b; b = c; sgn = -1.0f; }
    o = (a == 0) ? b - 1 : (a == 1 ? b + 1 : 5);
}
// channel comp 0..5 in the frame of charge axis mu (S8(b)): (0,mu) (0,nu) (0,rho) (nu,rho) (rho,mu) (mu,nu)
__device__ __forceinline__ void comp_dirs(int mu, int comp, int& a, int& b) {
    const int nu = 1 + (mu % 3), rho = 1 + ((mu + 1) % 3);
    switch (comp) {
        case 0: a = 0; b = mu; break;
        case 1: a = 0; b = nu; break;
        case 2: a = 0; b = rho; break;
        case 3: a = nu; b = rho; break;
        case 4: a = rho; b = mu; break;
        default: a = mu; b = nu; break;
    }
}

struct AccumArgs {
    Geom g;
    int d, n_slab, r_max, n_fp;
    int nk;               // configurations in this batch (1..KB), slots 0..nk-1 in sub-update order
    int r_begin, r_end;   // separations handled by this launch (multihit: r = 1 from the plain table, r >= 2 from Um)
    int a_r_max;          // the sums of T are written only for r <= a_r_max (field launch with multihit: r = 1 only)
    int first;            // 1: first pass of a measurement: the sums start from zero (no read, no memset)
    long long idx0, n_idx; // (s, xs) entries handled by this launch: [idx0, idx0 + n_idx)  (a range of slabs)
    const double2* U;     // [nk][n_slab*Vs]
    const float* Ot;      // [nk][12][n_slab*Vs]   (n_fp > 0 only)
    const int* fps;       // device int[n_fp][3]
    double2* A;
    double2* B;
};

// rows a7, a8 for a BATCH of nk <= KB configurations: one thread per (s, xs) loops over the charge axis mu and
// the separation r, reads each accumulator entry once, adds the nk terms in sub-update order (the same
// sequence of fp64 additions as nk single passes, so the result does not depend on the batching) and
// writes it back once: 32/nk bytes of accumulator traffic per entry and sub-update instead of 32.
// The accumulators are streamed (ld.cs / st.cs, RB entries in flight per thread); the U tables, which every
// site re-reads 6 r_max times, stay in L1/L2.
#ifndef UL_ACC_RB
#define UL_ACC_RB 2
#endif
#ifndef UL_ACCF_MINB
#define UL_ACCF_MINB 1
#endif
#ifndef UL_ACC_MINB
#define UL_ACC_MINB 3
#endif
constexpr int ACC_RB = UL_ACC_RB;

template <int KB, bool FIELD, bool FULL>
__global__ void __launch_bounds__(256, FIELD ? UL_ACCF_MINB : UL_ACC_MINB) k_accumulate(const AccumArgs P) {
    const Geom& g = P.g;
    const long long n = (long long)P.n_slab * g.Vs;
    const long long idx = P.idx0 + (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= P.idx0 + P.n_idx) return;
    const int s = (int)(idx / g.Vs);
    const int xs_lin = (int)(idx - (long long)s * g.Vs);
    const int Ns = g.Ns;
    const int stride[4] = {0, 1, Ns, Ns * Ns};
    const double2* __restrict__ Us = P.U + (long long)s * g.Vs;
    const long long stepA = (long long)P.n_slab * g.Vs;                  // A[mu][r] -> A[mu][r+1]
#pragma unroll
    for (int mu = 1; mu <= 3; ++mu) {
        const int nu = 1 + (mu % 3), rho = 1 + ((mu + 1) % 3);
        // The site this thread owns for the charge axis mu.  For mu = 3 it is the thread's linear site with x2 and x3 exchanged
        // (a bijection of the slab's sites), so that the consecutive x2 rows of a thread block become consecutive x3 rows: the
        // rows U(x + r 3^) a block reads are then shared between its rows through L1, as they are for mu = 2 (without the
        // exchange every one of them is read from L2 once per row and separation: half of the kernel's L2 traffic).  Every
        // accumulator entry still sees the same additions in the same order.
        int x[4];
        x[0] = 0;
        x[1] = xs_lin % Ns;
        x[2] = (xs_lin / Ns) % Ns;
        x[3] = xs_lin / (Ns * Ns);
        if (mu == 3) { const int t_ = x[2]; x[2] = x[3]; x[3] = t_; }
        const int xs = x[1] + Ns * (x[2] + Ns * x[3]);
        double2 u0[KB];
#pragma unroll
        for (int k = 0; k < KB; ++k)
            if (FULL || k < P.nk) u0[k] = Us[k * n + xs];
        double2* Ap = P.A + (((long long)(mu - 1) * P.r_max + (P.r_begin - 1)) * P.n_slab + s) * g.Vs + xs;
        // the accumulator entries of the NEXT step are requested before the current ones are worked on (software pipelining:
        // the kernel is bound by the latency of these reads, not by bandwidth or arithmetic)
        double2 an[ACC_RB];
#pragma unroll
        for (int i = 0; i < ACC_RB; ++i)
            an[i] = (P.first || P.r_begin + i > P.r_end || P.r_begin + i > P.a_r_max) ? make_double2(0.0, 0.0) : __ldcs(Ap + i * stepA);
        for (int r0 = P.r_begin; r0 <= P.r_end; r0 += ACC_RB) {
            double2 a[ACC_RB];
#pragma unroll
            for (int i = 0; i < ACC_RB; ++i) {
                a[i] = an[i];
                const int rn = r0 + ACC_RB + i;
                an[i] = (P.first || rn > P.r_end || rn > P.a_r_max) ? make_double2(0.0, 0.0) : __ldcs(Ap + (ACC_RB + i) * stepA);
            }
#pragma unroll
            for (int i = 0; i < ACC_RB; ++i) {
                const int r = r0 + i;
                if (r > P.r_end) break;
                // T^(d)(x,s,r mu) = U(x + r mu) conj(U(x))  (Eqs. 22, 25)
                const int ys = xs + (wrapc(x[mu] + r, Ns) - x[mu]) * stride[mu];         // r <= Ns/2
                double2 T[KB], v[KB];
#pragma unroll
                for (int k = 0; k < KB; ++k)                       // all loads of this entry in flight before the first use
                    if (FULL || k < P.nk) v[k] = Us[k * n + ys];
#pragma unroll
                for (int k = 0; k < KB; ++k)
                    if (FULL || k < P.nk) {
                        if (FIELD) {                               // T itself is needed for the TO sums
                            T[k].x = fma(v[k].x, u0[k].x, v[k].y * u0[k].y);
                            T[k].y = fma(v[k].y, u0[k].x, -(v[k].x * u0[k].y));
                        }
                        // the term folded into the sum (4 DFMA); the same arithmetic with and without field points,
                        // so the slab sums of T do not depend on what else is measured
                        a[i].x = fma(v[k].y, u0[k].y, fma(v[k].x, u0[k].x, a[i].x));
                        a[i].y = fma(-v[k].x, u0[k].y, fma(v[k].y, u0[k].x, a[i].y));
                    }
                if (r <= P.a_r_max) __stcs(Ap + i * stepA, a[i]);
                if (FIELD) {
                    for (int fp = 0; fp < P.n_fp; ++fp) {
                        // anchor y = x + (floor(r/2)+a) mu + b nu + c rho  (DESIGN R10)
                        int z[4] = {0, x[1], x[2], x[3]};
                        z[mu] = modc(z[mu] + r / 2 + P.fps[3 * fp], Ns);
                        z[nu] = modc(z[nu] + P.fps[3 * fp + 1], Ns);
                        z[rho] = modc(z[rho] + P.fps[3 * fp + 2], Ns);
                        const long long zs = z[1] + (long long)Ns * (z[2] + (long long)Ns * z[3]) + (long long)s * g.Vs;
                        const long long b_base = (((long long)(mu - 1) * P.r_max + (r - 1)) * P.n_slab + s) * P.n_fp + fp;
#pragma unroll
                        for (int comp = 0; comp < 6; ++comp) {
                            int pa, pb, o;
                            float sgn;
                            comp_dirs(mu, comp, pa, pb);
                            orient_of(pa, pb, o, sgn);
                            const long long b0 = (b_base * 12 + 2 * comp) * g.Vs + xs;
                            double2 bc = make_double2(0.0, 0.0), bs = make_double2(0.0, 0.0);
                            if (!P.first) { bc = __ldcs(P.B + b0); bs = __ldcs(P.B + b0 + g.Vs); }
#pragma unroll
                            for (int k = 0; k < KB; ++k)
                                if (FULL || k < P.nk) {
                                    const float* Otk = P.Ot + (long long)k * 12 * n;
                                    const double Oc = (double)Otk[(long long)(2 * o) * n + zs];
                                    const double Os = (double)(sgn * Otk[(long long)(2 * o + 1) * n + zs]);
                                    bc.x += T[k].x * Oc; bc.y += T[k].y * Oc;
                                    bs.x += T[k].x * Os; bs.y += T[k].y * Os;
                                }
                            __stcs(P.B + b0, bc);
                            __stcs(P.B + b0 + g.Vs, bs);
                        }
                    }
                }
            }
            Ap += ACC_RB * stepA;
        }
    }
}

// ---------------------------------------------------------------- two-level combine (row a9)
// A4[mu][r][S][xs] += prod_i [T](S m + i);  B4[..][S][fp][ch][xs] += sum_i [TO](i) prod_{i' != i} [T](i')
// with [.] = inner sum * inv.  One thread per (mu, r, S, xs).
struct CombineArgs {
    long long Vs;
    int r_max, n_fp, n_inner, n_outer, m;
    double inv;
    const double2* A2;
    const double2* B2;
    double2* A4;
    double2* B4;
};
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

__global__ void __launch_bounds__(256) k_combine(const CombineArgs P) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = 3LL * P.r_max * P.n_outer * P.Vs;
    if (idx >= total) return;
    const long long xs = idx % P.Vs;
    long long q = idx / P.Vs;
    const int S = (int)(q % P.n_outer);
    const long long mr = q / P.n_outer;                                        // (mu-1)*r_max + (r-1)
    double2 p = make_double2(1.0, 0.0);
    for (int i = 0; i < P.m; ++i) {
        double2 a = P.A2[(mr * P.n_inner + (long long)S * P.m + i) * P.Vs + xs];
        a.x *= P.inv; a.y *= P.inv;
        p = cmul(p, a);
    }
    double2 acc = P.A4[idx];
    acc.x += p.x; acc.y += p.y;
    P.A4[idx] = acc;
    for (int f = 0; f < P.n_fp * 12; ++f) {
        // dual-number product: prod_i (T_i + eps TO_i) = p + eps g
        double2 pp = make_double2(1.0, 0.0), gg = make_double2(0.0, 0.0);
        for (int i = 0; i < P.m; ++i) {
            const long long si = mr * P.n_inner + (long long)S * P.m + i;
            double2 a = P.A2[si * P.Vs + xs];
            double2 b = P.B2[(si * (P.n_fp * 12) + f) * P.Vs + xs];
            a.x *= P.inv; a.y *= P.inv; b.x *= P.inv; b.y *= P.inv;
            const double2 g1 = cmul(gg, a), g2 = cmul(pp, b);
            gg = make_double2(g1.x + g2.x, g1.y + g2.y);
            pp = cmul(pp, a);
        }
        const long long o = ((mr * P.n_outer + S) * (P.n_fp * 12) + f) * P.Vs + xs;
        double2 b4 = P.B4[o];
        b4.x += gg.x; b4.y += gg.y;
        P.B4[o] = b4;
    }
}

// ---------------------------------------------------------------- slab product + lattice sum (row a10)
// output o < r_max:            C(r)        = sum_{mu,xs} prod_s [T](s)
// output o = r_max + (r-1)*12F + f:  G(r,f) = sum_{mu,xs} sum_s [TO](s) prod_{s' != s} [T](s')
// partial[(2*o + reim)*nblk + b]
struct ReduceArgs {
    long long Vs;
    int r_max, n_fp, n_slab;
    double inv;
    const double2* A;
    const double2* B;
    double* partial;
};
template <bool FIELD>
__global__ void __launch_bounds__(256) k_slab_product(const ReduceArgs P, int o_first) {
    __shared__ double sm[2 * 32];
    const int o = o_first + blockIdx.y;
    const int F12 = P.n_fp * 12;
    const int r1 = FIELD ? (o - P.r_max) / F12 : o;                            // r - 1
    const int f = FIELD ? (o - P.r_max) - r1 * F12 : 0;
    double v[2] = {0.0, 0.0};
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < 3 * P.Vs; j += (long long)gridDim.x * blockDim.x) {
        const int mu1 = (int)(j / P.Vs);
        const long long xs = j - (long long)mu1 * P.Vs;
        const long long mr = (long long)mu1 * P.r_max + r1;
        const double2* Ap = P.A + mr * P.n_slab * P.Vs + xs;
        double2 pp = make_double2(1.0, 0.0), gg = make_double2(0.0, 0.0);
        if (!FIELD) {
            int s = 0;
            for (; s + 4 <= P.n_slab; s += 4) {                                 // four loads in flight per thread
                double2 a[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) a[i] = __ldcs(Ap + (long long)(s + i) * P.Vs);
#pragma unroll
                for (int i = 0; i < 4; ++i) { a[i].x *= P.inv; a[i].y *= P.inv; pp = cmul(pp, a[i]); }
            }
            for (; s < P.n_slab; ++s) {
                double2 a = __ldcs(Ap + (long long)s * P.Vs);
                a.x *= P.inv; a.y *= P.inv;
                pp = cmul(pp, a);
            }
            v[0] += pp.x; v[1] += pp.y;
        } else {
            for (int s = 0; s < P.n_slab; ++s) {
                const long long si = mr * P.n_slab + s;
                double2 a = Ap[(long long)s * P.Vs];
                double2 b = P.B[(si * F12 + f) * P.Vs + xs];
                a.x *= P.inv; a.y *= P.inv; b.x *= P.inv; b.y *= P.inv;
                const double2 g1 = cmul(gg, a), g2 = cmul(pp, b);
                gg = make_double2(g1.x + g2.x, g1.y + g2.y);
                pp = cmul(pp, a);
            }
            v[0] += gg.x; v[1] += gg.y;
        }
    }
    block_sum<2>(v, sm);
    if (threadIdx.x == 0) {
        P.partial[(long long)(2 * o) * gridDim.x + blockIdx.x] = v[0];
        P.partial[(long long)(2 * o + 1) * gridDim.x + blockIdx.x] = v[1];
    }
}

// ---------------------------------------------------------------- replay estimator of the field correlators
// The estimator G(r,fp,ch) = (1/(3 Vs Nt)) sum_{x,mu,s} [TO](x,s) prod_{s' != s} [T](x,s')  (Eq. 34) is linear
// in O, and the sub-update trajectory can be replayed bit for bit (counter-based RNG).  Pass 1 accumulates only the
// sums of T; k_slab_weights turns them into W(x,s,mu,r) = prod_{s' != s} [T](x,s'); pass 2 replays the sub-updates and
// k_replay_reduce adds sum_{x,mu,s} W T_j sum_{t in slab} O_ch(x + off) of every configuration j straight into
// lattice sums: no per-site TO accumulators (12 n_fp times the memory and traffic of the T accumulators).
struct WeightArgs {
    long long Vs;
    int r_max, n_slab;
    double inv;           // 1 / n_sub
    const double2* A;     // sums of T, [mu][r][s][xs]
    double2* W;           // out, same layout
};
__global__ void __launch_bounds__(256) k_slab_weights(const WeightArgs P) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;            // over (mu, r, xs)
    if (idx >= 3LL * P.r_max * P.Vs) return;
    const long long mr = idx / P.Vs, xs = idx - mr * P.Vs;
    const double2* Ap = P.A + mr * P.n_slab * P.Vs + xs;
    double2* Wp = P.W + mr * P.n_slab * P.Vs + xs;
    double2 run = make_double2(1.0, 0.0);
    for (int s = 0; s < P.n_slab; ++s) {                                                // prefix products
        Wp[(long long)s * P.Vs] = run;
        double2 a = Ap[(long long)s * P.Vs];
        a.x *= P.inv; a.y *= P.inv;
        run = cmul(run, a);
    }
    run = make_double2(1.0, 0.0);
    for (int s = P.n_slab - 1; s >= 0; --s) {                                           // times suffix products
        Wp[(long long)s * P.Vs] = cmul(Wp[(long long)s * P.Vs], run);
        double2 a = Ap[(long long)s * P.Vs];
        a.x *= P.inv; a.y *= P.inv;
        run = cmul(run, a);
    }
}

// product of the slab averages [T](x,s) over the slabs s_begin <= s < s_end, per (mu, r, xs): the piece of the slab
// product (row a10) that one shard of a t-partitioned lattice owns
__global__ void __launch_bounds__(256) k_slab_partial_product(const WeightArgs P, int s_begin, int s_end) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;            // over (mu, r, xs)
    if (idx >= 3LL * P.r_max * P.Vs) return;
    const long long mr = idx / P.Vs, xs = idx - mr * P.Vs;
    const double2* Ap = P.A + mr * P.n_slab * P.Vs + xs;
    double2 run = make_double2(1.0, 0.0);
    for (int s = s_begin; s < s_end; ++s) {
        double2 a = Ap[(long long)s * P.Vs];
        a.x *= P.inv; a.y *= P.inv;
        run = cmul(run, a);
    }
    P.W[idx] = run;
}

// The shards' partial products multiplied in rank order and summed over the lattice and the three directions: the last
// step of row a10 for a t-partitioned lattice (Eq. 24, Eq. 26).  part[k] = shard k's
// [mu][r][xs] array (k_slab_partial_product; the own one or a copy received from rank k).  Grid (blocks, r_max);
// partial[(2*(r-1) + reim)*gridDim.x + b], the layout k_sum_partials reads: a fixed two-stage tree.
constexpr int MAX_SHARDS = 64;
struct CombinePartsArgs {
    long long Vs;
    int r_max, n_parts;
    const double2* part[MAX_SHARDS];
    double* partial;
};
__global__ void __launch_bounds__(256) k_combine_partial_products(const CombinePartsArgs P) {
    __shared__ double sm[2 * 32];
    const int r1 = blockIdx.y;
    double v[2] = {0.0, 0.0};
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < 3 * P.Vs; j += (long long)gridDim.x * blockDim.x) {
        const int mu1 = (int)(j / P.Vs);
        const long long idx = ((long long)mu1 * P.r_max + r1) * P.Vs + (j - (long long)mu1 * P.Vs);
        double2 pp = P.part[0][idx];
        for (int k = 1; k < P.n_parts; ++k) pp = cmul(pp, P.part[k][idx]);
        v[0] += pp.x; v[1] += pp.y;
    }
    block_sum<2>(v, sm);
    if (threadIdx.x == 0) {
        P.partial[(long long)(2 * r1) * gridDim.x + blockIdx.x] = v[0];
        P.partial[(long long)(2 * r1 + 1) * gridDim.x + blockIdx.x] = v[1];
    }
}

// Two-level replay weights: for the inner slab s = S m + i of outer slab S,
//   Wc(x,s) = W4(x,S) prod_{i' != i} [T2](x, S m + i'),  W4(x,S) = prod_{S' != S} [T4](x,S')   (Eqs. 32-34 with the TO term
// factored out: G is linear in O), [T2] = A2 * inv (inner sums of THIS outer iteration).  One thread per (mu, r, xs).
struct GroupWeightArgs {
    long long Vs;
    int r_max, n_inner, n_outer, m;
    double inv;           // 1 / n_in
    const double2* A2;    // [mu][r][n_inner][xs]
    const double2* W4;    // [mu][r][n_outer][xs]
    double2* Wc;          // out [mu][r][n_inner][xs]
};
__global__ void __launch_bounds__(256) k_group_weights(const GroupWeightArgs P) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 3LL * P.r_max * P.Vs) return;
    const long long mr = idx / P.Vs, xs = idx - mr * P.Vs;
    const double2* Ap = P.A2 + mr * P.n_inner * P.Vs + xs;
    double2* Wp = P.Wc + mr * P.n_inner * P.Vs + xs;
    for (int S = 0; S < P.n_outer; ++S) {
        const double2 w4 = P.W4[(mr * P.n_outer + S) * P.Vs + xs];
        double2 run = w4;
        for (int i = 0; i < P.m; ++i) {                                                 // W4 times the prefix products
            const long long s = (long long)S * P.m + i;
            Wp[s * P.Vs] = run;
            double2 a = Ap[s * P.Vs];
            a.x *= P.inv; a.y *= P.inv;
            run = cmul(run, a);
        }
        run = make_double2(1.0, 0.0);
        for (int i = P.m - 1; i >= 0; --i) {                                            // times the suffix products
            const long long s = (long long)S * P.m + i;
            Wp[s * P.Vs] = cmul(Wp[s * P.Vs], run);
            double2 a = Ap[s * P.Vs];
            a.x *= P.inv; a.y *= P.inv;
            run = cmul(run, a);
        }
    }
}

struct ReplayArgs {
    Geom g;
    int n_slab, r_max, n_fp;
    const double2* U;     // [n_slab*Vs]  this configuration
    const float* Ot;      // [12][n_slab*Vs]
    const int* fps;
    const double2* W;
    double* partial;      // [(2*o + reim)*gridDim.x + b], o = r_max + ((r-1)*n_fp + fp)*12 + ch  (the layout of k_slab_product)
};
// grid (nblk, r_max * n_fp): block (b, e) sums its share of the sites for separation r = e / n_fp + 1, field point e % n_fp
__global__ void __launch_bounds__(256) k_replay_reduce(const ReplayArgs P) {
    __shared__ double sm[24 * 32];
    const Geom& g = P.g;
    const int Ns = g.Ns;
    const int r = blockIdx.y / P.n_fp + 1, fp = blockIdx.y - (r - 1) * P.n_fp;
    const long long n = (long long)P.n_slab * g.Vs;
    const int fa = P.fps[3 * fp], fb = P.fps[3 * fp + 1], fc = P.fps[3 * fp + 2];
    double acc[24];
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0.0;
    const int stride[4] = {0, 1, Ns, Ns * Ns};
#pragma unroll
    for (int mu = 1; mu <= 3; ++mu) {
        const int nu = 1 + (mu % 3), rho = 1 + ((mu + 1) % 3);
        const double2* Wm = P.W + ((long long)(mu - 1) * P.r_max + (r - 1)) * n;
        for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) {
            const int s = (int)(j / g.Vs);
            const int xs = (int)(j - (long long)s * g.Vs);
            int x[4] = {0, xs % Ns, (xs / Ns) % Ns, xs / (Ns * Ns)};
            const int ys = xs + (wrapc(x[mu] + r, Ns) - x[mu]) * stride[mu];
            const double2 u = P.U[j], v = P.U[(long long)s * g.Vs + ys], w = Wm[j];
            const double2 T = make_double2(fma(v.x, u.x, v.y * u.y), fma(v.y, u.x, -(v.x * u.y)));   // U(x + r mu) conj U(x)
            const double2 Z = cmul(w, T);
            int z[4] = {0, x[1], x[2], x[3]};
            z[mu] = modc(z[mu] + r / 2 + fa, Ns);                                        // anchor, DESIGN R10
            z[nu] = modc(z[nu] + fb, Ns);
            z[rho] = modc(z[rho] + fc, Ns);
            const long long zs = z[1] + (long long)Ns * (z[2] + (long long)Ns * z[3]) + (long long)s * g.Vs;
#pragma unroll
            for (int comp = 0; comp < 6; ++comp) {
                int pa, pb, o;
                float sgn;
                comp_dirs(mu, comp, pa, pb);
                orient_of(pa, pb, o, sgn);
                const double Oc = (double)P.Ot[(long long)(2 * o) * n + zs];
                const double Os = (double)(sgn * P.Ot[(long long)(2 * o + 1) * n + zs]);
                acc[4 * comp + 0] = fma(Z.x, Oc, acc[4 * comp + 0]);
                acc[4 * comp + 1] = fma(Z.y, Oc, acc[4 * comp + 1]);
                acc[4 * comp + 2] = fma(Z.x, Os, acc[4 * comp + 2]);
                acc[4 * comp + 3] = fma(Z.y, Os, acc[4 * comp + 3]);
            }
        }
    }
    block_sum<24>(acc, sm);
    if (threadIdx.x == 0) {
        const long long o0 = P.r_max + ((long long)(r - 1) * P.n_fp + fp) * 12;          // ch = 2 comp + kind; acc = [ch][reim]
#pragma unroll
        for (int i = 0; i < 24; ++i) P.partial[(2 * (o0 + i / 2) + (i & 1)) * gridDim.x + blockIdx.x] = acc[i];
    }
}

constexpr int PLANE_MAX_NS = 64;   // the DFT route keeps three Ns^2 planes of complex doubles in shared memory (196 KB at Ns = 64)

// ---------------------------------------------------------------- full-plane maps through the transverse DFT
// When the field points are a FULL transverse plane, fp = b + Ns c <-> offset (a, b, c) with one a (BJ config 4's "full
// mid-plane maps"), the map of one lattice plane (s, x_mu) is a 2-d cross-correlation, Z = W T on the plane x_mu, O on the
// plane x_mu + floor(r/2) + a:
// G(b,c) = sum_{p,q} Z(p,q) O(p+b, q+c)  <=>  Ghat(k,l) = Zhat(-k,-l) Ohat(k,l)  with the 2-d DFT over the transverse plane:
// 2 Ns^3 complex MACs per plane for the transforms instead of Ns^4 per plane and channel for the direct sum.  The DFT is
// done as two small dense matrix products with the Ns x Ns matrix W[j][k] = e^{-2 pi i jk/Ns} (any Ns, no radix
// restriction), in fp64, one thread block per plane whose threads own EPT = 1, 2 or 4 entries each (Ns^2 / EPT <= 1024
// threads: Ns <= 64).  Ohat of the 12 channels of one direction mu is tabulated first (k_plane_dft_o); k_plane_spectral
// transforms Z = W T of every plane of its group, multiplies with CHB = 6 / EPT (at least 1) of the 12 Ohat planes and keeps
// those complex sums per (k,l) in registers; k_plane_gh_accum adds the groups' partial sums to Ghat; k_plane_idft turns
// Ghat into the map once per measurement.  Everything is owned by one thread per entry and summed in a fixed order:
// bitwise reproducible.
__device__ __forceinline__ void dft_matrix_to_smem(double2* Wm, int Ns, bool conjugate) {
    for (int e = threadIdx.x; e < Ns * Ns; e += blockDim.x) {
        const int j = e / Ns, k = e - j * Ns;
        double sn, cs;
        sincospi(2.0 * (double)((j * k) % Ns) / (double)Ns, &sn, &cs);
        Wm[e] = make_double2(cs, conjugate ? sn : -sn);
    }
}
// Ahat = M A M for the plane in A; M symmetric; T is scratch.  Thread x owns the entries e = x + i blockDim.x, i < EPT
// (e = k*Ns + l); their values are returned in r[].
template <int EPT>
__device__ __forceinline__ void dft2_entries(const double2* A, double2* T, const double2* M, int Ns, double2 r[EPT]) {
#pragma unroll
    for (int i = 0; i < EPT; ++i) {
        const int e = threadIdx.x + i * blockDim.x, k = e / Ns, l = e - k * Ns;
        double2 t = make_double2(0.0, 0.0);
        for (int p = 0; p < Ns; ++p) {                                   // T[k][l] = sum_p M[k][p] A[p][l]
            const double2 m = M[k * Ns + p], a = A[p * Ns + l];
            t.x = fma(m.x, a.x, fma(-m.y, a.y, t.x));
            t.y = fma(m.x, a.y, fma(m.y, a.x, t.y));
        }
        T[e] = t;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < EPT; ++i) {
        const int e = threadIdx.x + i * blockDim.x, k = e / Ns, l = e - k * Ns;
        double2 v = make_double2(0.0, 0.0);
        for (int q = 0; q < Ns; ++q) {                                   // R[k][l] = sum_q T[k][q] M[q][l]
            const double2 a = T[k * Ns + q], m = M[q * Ns + l];
            v.x = fma(a.x, m.x, fma(-a.y, m.y, v.x));
            v.y = fma(a.x, m.y, fma(a.y, m.x, v.y));
        }
        r[i] = v;
    }
    __syncthreads();
}

// Ohat[ch][plane][k*Ns + l] for direction mu; grid (n_planes, 12), block Ns^2 / EPT, dynamic smem 3 Ns^2 double2
template <int EPT>
__global__ void __launch_bounds__(1024, 1) k_plane_dft_o(const ReplayArgs P, int mu, double2* __restrict__ Oh) {
    extern __shared__ double2 sh[];
    const Geom& g = P.g;
    const int Ns = g.Ns, N2 = Ns * Ns;
    double2 *Wm = sh, *A = sh + N2, *T = sh + 2 * N2;
    const int nu = 1 + (mu % 3), rho = 1 + ((mu + 1) % 3);
    const int stride[4] = {0, 1, Ns, Ns * Ns};
    const long long n = (long long)P.n_slab * g.Vs;
    const int pl = blockIdx.x, s = pl / Ns, xm = pl - s * Ns, ch = blockIdx.y;
    int pa, pb, o;
    float sgn;
    comp_dirs(mu, ch >> 1, pa, pb);
    orient_of(pa, pb, o, sgn);
    dft_matrix_to_smem(Wm, Ns, false);
#pragma unroll
    for (int i = 0; i < EPT; ++i) {
        const int e = threadIdx.x + i * blockDim.x, p = e / Ns, q = e - p * Ns;
        const long long zs = (long long)s * g.Vs + xm * stride[mu] + p * stride[nu] + q * stride[rho];
        const float v = P.Ot[(long long)(2 * o + (ch & 1)) * n + zs];
        A[e] = make_double2((double)((ch & 1) ? sgn * v : v), 0.0);
    }
    __syncthreads();
    double2 r[EPT];
    dft2_entries<EPT>(A, T, Wm, Ns, r);
#pragma unroll
    for (int i = 0; i < EPT; ++i) Oh[((long long)ch * gridDim.x + pl) * N2 + threadIdx.x + i * blockDim.x] = r[i];
}

// partial[(group*r_max + r-1)*12 + ch][k*Ns + l] = sum over the planes of the group of Zhat(-k,-l) Ohat_ch(k,l);
// grid (r_max, groups, 12 / CHB), block Ns^2 / EPT (<= 1024 threads with 64 registers each: CHB * EPT <= 6 complex sums)
template <int EPT>
__global__ void __launch_bounds__(1024, 1) k_plane_spectral(const ReplayArgs P, int mu, int fa, const double2* __restrict__ Oh, double2* __restrict__ Ghp) {
    constexpr int CHB = EPT >= 4 ? 1 : 6 / EPT;
    extern __shared__ double2 sh[];
    const Geom& g = P.g;
    const int Ns = g.Ns, N2 = Ns * Ns;
    double2 *Wc = sh, *A = sh + N2, *T = sh + 2 * N2;
    const int nu = 1 + (mu % 3), rho = 1 + ((mu + 1) % 3);
    const int stride[4] = {0, 1, Ns, Ns * Ns};
    const long long n = (long long)P.n_slab * g.Vs;
    const int r = blockIdx.x + 1, n_planes = P.n_slab * Ns;
    const double2* Wm = P.W + ((long long)(mu - 1) * P.r_max + (r - 1)) * n;
    dft_matrix_to_smem(Wc, Ns, true);                                    // conj(W): Zhat(-k,-l)
    const int ch0 = CHB * blockIdx.z;
    double2 acc[CHB][EPT];
#pragma unroll
    for (int ch = 0; ch < CHB; ++ch)
#pragma unroll
        for (int i = 0; i < EPT; ++i) acc[ch][i] = make_double2(0.0, 0.0);
    for (int pl = blockIdx.y; pl < n_planes; pl += gridDim.y) {
        const int s = pl / Ns, xm = pl - s * Ns;
#pragma unroll
        for (int i = 0; i < EPT; ++i) {
            const int e = threadIdx.x + i * blockDim.x, p = e / Ns, q = e - p * Ns;
            const int xs = xm * stride[mu] + p * stride[nu] + q * stride[rho];
            const int ys = wrapc(xm + r, Ns) * stride[mu] + p * stride[nu] + q * stride[rho];
            const long long j = (long long)s * g.Vs + xs;
            const double2 u = P.U[j], v = P.U[(long long)s * g.Vs + ys];
            const double2 Tj = make_double2(fma(v.x, u.x, v.y * u.y), fma(v.y, u.x, -(v.x * u.y)));
            A[e] = cmul(Wm[j], Tj);
        }
        __syncthreads();
        double2 zh[EPT];
        dft2_entries<EPT>(A, T, Wc, Ns, zh);
        const int plo = s * Ns + modc(xm + r / 2 + fa, Ns);              // plane of the plaquettes (anchor, DESIGN R10)
#pragma unroll
        for (int ch = 0; ch < CHB; ++ch)
#pragma unroll
            for (int i = 0; i < EPT; ++i) {
                const double2 oh = Oh[((long long)(ch0 + ch) * n_planes + plo) * N2 + threadIdx.x + i * blockDim.x];
                acc[ch][i].x = fma(zh[i].x, oh.x, fma(-zh[i].y, oh.y, acc[ch][i].x));
                acc[ch][i].y = fma(zh[i].x, oh.y, fma(zh[i].y, oh.x, acc[ch][i].y));
            }
    }
#pragma unroll
    for (int ch = 0; ch < CHB; ++ch)
#pragma unroll
        for (int i = 0; i < EPT; ++i)
            Ghp[(((long long)blockIdx.y * P.r_max + (r - 1)) * 12 + ch0 + ch) * N2 + threadIdx.x + i * blockDim.x] = acc[ch][i];
}

// Gh[(r-1)*12 + ch][kl] += sum_groups Ghp[group][...]; one thread per entry
__global__ void __launch_bounds__(256) k_plane_gh_accum(const double2* __restrict__ Ghp, int groups, long long n_entries, double2* __restrict__ Gh) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_entries) return;
    double2 a = Gh[i];
    for (int gidx = 0; gidx < groups; ++gidx) { const double2 v = Ghp[(long long)gidx * n_entries + i]; a.x += v.x; a.y += v.y; }
    Gh[i] = a;
}

// field[((r-1)*Ns^2 + (b + Ns c))*12 + ch] = scale/Ns^2 * sum_{k,l} Gh(k,l) e^{+2 pi i (kb + lc)/Ns}; grid (r_max, 12), block Ns^2 / EPT
template <int EPT>
__global__ void __launch_bounds__(1024, 1) k_plane_idft(const double2* __restrict__ Gh, int Ns, double scale, double2* __restrict__ field) {
    extern __shared__ double2 sh[];
    const int N2 = Ns * Ns;
    double2 *Wc = sh, *A = sh + N2, *T = sh + 2 * N2;
    const int r1 = blockIdx.x, ch = blockIdx.y;
    dft_matrix_to_smem(Wc, Ns, true);
#pragma unroll
    for (int i = 0; i < EPT; ++i) A[threadIdx.x + i * blockDim.x] = Gh[((long long)r1 * 12 + ch) * N2 + threadIdx.x + i * blockDim.x];
    __syncthreads();
    double2 v[EPT];
    dft2_entries<EPT>(A, T, Wc, Ns, v);                                  // entry e = b*Ns + c
    const double f = scale / (double)N2;
#pragma unroll
    for (int i = 0; i < EPT; ++i) {
        const int e = threadIdx.x + i * blockDim.x, b = e / Ns, c = e - b * Ns;
        field[((long long)r1 * N2 + (b + Ns * c)) * 12 + ch] = make_double2(v[i].x * f, v[i].y * f);
    }
}

// vacuum[ch] = (1/(3 V n_acc)) sum_mu sgn * colsum[orient(mu, comp)][kind]
__global__ void k_vacuum(const double* __restrict__ colsum /*[12]*/, double scale, double* __restrict__ vac /*[12]*/) {
    const int ch = threadIdx.x;
    if (ch >= 12) return;
    const int comp = ch >> 1, kind = ch & 1;
    double v = 0.0;
    for (int mu = 1; mu <= 3; ++mu) {
        int a, b, o;
        float sgn;
        comp_dirs(mu, comp, a, b);
        orient_of(a, b, o, sgn);
        v += (kind ? (double)sgn : 1.0) * colsum[2 * o + kind];
    }
    vac[ch] = v * scale;
}

}  // namespace ulk
