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
// theta_P(a,b)(y) = theta_a(y) + theta_b(y+a) - theta_a(y+b) - theta_b(y), binary angle (exact mod 2 pi)
__device__ __forceinline__ int plaq_fx(const Geom& g, const int* __restrict__ th, int a, int b, const int x[4]) {
    int xa[4] = {x[0], x[1], x[2], x[3]}, xb[4] = {x[0], x[1], x[2], x[3]};
    xa[a] = (x[a] + 1 == (a == 0 ? g.Nt : g.Ns)) ? 0 : x[a] + 1;
    xb[b] = (x[b] + 1 == (b == 0 ? g.Nt : g.Ns)) ? 0 : x[b] + 1;
    const unsigned t0 = (unsigned)__ldg(th + link_index(g, a, x[0], x[3], x[2], x[1]));
    const unsigned t1 = (unsigned)__ldg(th + link_index(g, b, xa[0], xa[3], xa[2], xa[1]));
    const unsigned t2 = (unsigned)__ldg(th + link_index(g, a, xb[0], xb[3], xb[2], xb[1]));
    const unsigned t3 = (unsigned)__ldg(th + link_index(g, b, x[0], x[3], x[2], x[1]));
    return (int)(t0 + t1 - t2 - t3);
}

// row a11: partial[0*nblk + b] = sum of cos over time-like plaquettes, [1*nblk + b] space-like
__global__ void __launch_bounds__(256) k_plaquette(Geom g, const int* __restrict__ th, double* __restrict__ partial) {
    __shared__ double sm[2 * 32];
    double v[2] = {0.0, 0.0};
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.V; i += (long long)gridDim.x * blockDim.x) {
        long long s = i;
        int x[4];
        x[1] = (int)(s % g.Ns); s /= g.Ns;
        x[2] = (int)(s % g.Ns); s /= g.Ns;
        x[3] = (int)(s % g.Ns); s /= g.Ns;
        x[0] = (int)s;
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = a + 1; b < 4; ++b) {
                float c, sn;
                ulm::sincos_bt(plaq_fx(g, th, a, b, x), c, sn);
                if (a == 0) v[0] += (double)c; else v[1] += (double)c;
            }
    }
    block_sum<2>(v, sm);
    if (threadIdx.x == 0) { partial[blockIdx.x] = v[0]; partial[gridDim.x + blockIdx.x] = v[1]; }
}

// ---------------------------------------------------------------- per-configuration slab tables
// Th[s][xs] = sum_{t in slab s} theta_0(xs,t), binary angle (wrapping sum = exact mod 2 pi)
// Ot[o][kind][s][xs] = sum_{t in slab s} O(theta_P(o)(xs,t)),  O = 1 - cos (kind 0), sin (kind 1)
__global__ void __launch_bounds__(256) k_slab_tables(Geom g, const int* __restrict__ th, int d, int n_slab,
                                                     int* __restrict__ Th, float* __restrict__ Ot) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)n_slab * g.Vs) return;
    const int s = (int)(idx / g.Vs);
    long long r = idx - (long long)s * g.Vs;
    int x[4];
    x[1] = (int)(r % g.Ns); r /= g.Ns;
    x[2] = (int)(r % g.Ns); r /= g.Ns;
    x[3] = (int)r;
    unsigned acc = 0u;
    float o_c[6], o_s[6];
#pragma unroll
    for (int o = 0; o < 6; ++o) { o_c[o] = 0.0f; o_s[o] = 0.0f; }
    for (int t = s * d; t < (s + 1) * d; ++t) {
        x[0] = t;
        acc += (unsigned)__ldg(th + link_index(g, 0, t, x[3], x[2], x[1]));
        int o = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = a + 1; b < 4; ++b) {
                float c, sn;
                ulm::sincos_bt(plaq_fx(g, th, a, b, x), c, sn);
                o_c[o] += 1.0f - c;
                o_s[o] += sn;
                ++o;
            }
    }
    Th[idx] = (int)acc;
    const long long stride = (long long)n_slab * g.Vs;
#pragma unroll
    for (int o = 0; o < 6; ++o) {
        Ot[(long long)(2 * o) * stride + idx] = o_c[o];
        Ot[(long long)(2 * o + 1) * stride + idx] = o_s[o];
    }
}

// column sums of Ot for the vacuum expectation values: partial[col*nblk + b], col = 2*o + kind
__global__ void __launch_bounds__(256) k_ot_colsum(const float* __restrict__ Ot, long long n, double* __restrict__ partial) {
    __shared__ double sm[32];
    const int col = blockIdx.y;
    double v[1] = {0.0};
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        v[0] += (double)Ot[(long long)col * n + i];
    block_sum<1>(v, sm);
    if (threadIdx.x == 0) partial[(long long)col * gridDim.x + blockIdx.x] = v[0];
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
    const int* Th;
    const float* Ot;
    const int* fps;       // device int[n_fp][3]
    double2* A;
    double2* B;
};

// rows a7, a8: one thread per (s, xs); loops over the charge axis mu and separation r
__global__ void __launch_bounds__(256) k_accumulate(const AccumArgs P) {
    const Geom& g = P.g;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)P.n_slab * g.Vs) return;
    const int s = (int)(idx / g.Vs);
    const long long xs = idx - (long long)s * g.Vs;
    long long q = xs;
    int x[4];
    x[0] = 0;
    x[1] = (int)(q % g.Ns); q /= g.Ns;
    x[2] = (int)(q % g.Ns); q /= g.Ns;
    x[3] = (int)q;
    const int Ns = g.Ns;
    const int* Ths = P.Th + (long long)s * g.Vs;
    const int th0 = Ths[xs];
    const long long ot_stride = (long long)P.n_slab * g.Vs;
    for (int mu = 1; mu <= 3; ++mu) {
        const int nu = 1 + (mu % 3), rho = 1 + ((mu + 1) % 3);
        for (int r = 1; r <= P.r_max; ++r) {
            int y[4] = {0, x[1], x[2], x[3]};
            y[mu] = wrapc(x[mu] + r, Ns);                                      // r <= Ns/2
            const long long ys = y[1] + (long long)Ns * (y[2] + (long long)Ns * y[3]);
            // T^(d)(x,s,r mu) = exp(i sum_{t in slab} [theta_0(x + r mu, t) - theta_0(x, t)])  (Eq. 22, 25)
            float c, sn;
            ulm::sincos_bt((int)((unsigned)Ths[ys] - (unsigned)th0), c, sn);
            const double Tr = (double)c, Ti = (double)sn;
            const long long a_idx = (((long long)(mu - 1) * P.r_max + (r - 1)) * P.n_slab + s) * g.Vs + xs;
            double2 a = P.A[a_idx];
            a.x += Tr; a.y += Ti;
            P.A[a_idx] = a;
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
                    const double Oc = (double)P.Ot[(long long)(2 * o) * ot_stride + zs];
                    const double Os = (double)(sgn * P.Ot[(long long)(2 * o + 1) * ot_stride + zs]);
                    const long long b0 = (b_base * 12 + 2 * comp) * g.Vs + xs;
                    double2 b = P.B[b0];
                    b.x += Tr * Oc; b.y += Ti * Oc;
                    P.B[b0] = b;
                    b = P.B[b0 + g.Vs];
                    b.x += Tr * Os; b.y += Ti * Os;
                    P.B[b0 + g.Vs] = b;
                }
            }
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
__global__ void __launch_bounds__(256) k_slab_product(const ReduceArgs P) {
    __shared__ double sm[2 * 32];
    const int o = blockIdx.y;
    const int F12 = P.n_fp * 12;
    const bool is_c = o < P.r_max;
    const int r1 = is_c ? o : (o - P.r_max) / F12;                             // r - 1
    const int f = is_c ? 0 : (o - P.r_max) - r1 * F12;
    double v[2] = {0.0, 0.0};
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < 3 * P.Vs; j += (long long)gridDim.x * blockDim.x) {
        const int mu1 = (int)(j / P.Vs);
        const long long xs = j - (long long)mu1 * P.Vs;
        const long long mr = (long long)mu1 * P.r_max + r1;
        double2 pp = make_double2(1.0, 0.0), gg = make_double2(0.0, 0.0);
        for (int s = 0; s < P.n_slab; ++s) {
            const long long si = mr * P.n_slab + s;
            double2 a = P.A[si * P.Vs + xs];
            a.x *= P.inv; a.y *= P.inv;
            if (!is_c) {
                double2 b = P.B[(si * F12 + f) * P.Vs + xs];
                b.x *= P.inv; b.y *= P.inv;
                const double2 g1 = cmul(gg, a), g2 = cmul(pp, b);
                gg = make_double2(g1.x + g2.x, g1.y + g2.y);
            }
            pp = cmul(pp, a);
        }
        v[0] += is_c ? pp.x : gg.x;
        v[1] += is_c ? pp.y : gg.y;
    }
    block_sum<2>(v, sm);
    if (threadIdx.x == 0) {
        P.partial[(long long)(2 * o) * gridDim.x + blockIdx.x] = v[0];
        P.partial[(long long)(2 * o + 1) * gridDim.x + blockIdx.x] = v[1];
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
