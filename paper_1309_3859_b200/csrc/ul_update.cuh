// ul_update.cuh -- link-update kernels: staple gather + heatbath / overrelaxation sub-step,
// full or slab-masked.
//
// Layout (row a1, BJ kernel 1): th[mu][par][row*Nh + h], fp32 radians, where
//   row = (t*Ns + x3)*Ns + x2,  Nh = Ns/2,  par = (x1+x2+x3+t)&1,  x1 = 2h + ((par+x2+x3+t)&1).
// One sub-step (parity p, direction MU) updates the array th[MU][p] in place and reads the
// seven other arrays it depends on; it never reads an element another thread writes.
//
// Thread mapping: a thread owns VEC consecutive h of one row (VEC links).  Neighbours that are
// displaced in x2, x3, t keep the same h (aligned vector loads); a displacement in x1 shifts h
// by 0 or +-1 depending on the row's offset bit, which is handled with one extra scalar load.
#pragma once
#include "ul_math.cuh"

namespace ulk {

struct UpdateArgs {
    float* th;            // internal layout, 8 arrays of Vh floats
    long long Vh;         // V/2
    int Ns, Nh, Nt;
    int parity;           // sub-step parity p
    int slab_d;           // 0 = unmasked; else spatial links with t % slab_d == 0 are frozen
    float beta;
    uint32_t key0, key1;  // Philox key = seed
    uint32_t sweep_lo, sweep_hi;
};

// Loads, as fixed point, the VEC angles of the row at `rowp` that sit at x1-displacement D1
// (-1, 0, +1) from the thread's own sites h0..h0+VEC-1 with offset bit `off` (x1 = 2h + off):
// x1 + 1 lives at h + off, x1 - 1 at h - 1 + off of the other-parity row (periodic in Nh).
template <int VEC, int D1>
__device__ __forceinline__ void load_row(const float* __restrict__ rowp, int h0, int off, int Nh, int out[VEC]) {
    float v[VEC];
    if (VEC == 4) {
        const float4 q = __ldg(reinterpret_cast<const float4*>(rowp + h0));
        v[0] = q.x; v[1 % VEC] = q.y; v[2 % VEC] = q.z; v[3 % VEC] = q.w;
    } else if (VEC == 2) {
        const float2 q = __ldg(reinterpret_cast<const float2*>(rowp + h0));
        v[0] = q.x; v[1 % VEC] = q.y;
    } else {
        v[0] = __ldg(rowp + h0);
    }
    if (D1 > 0) {
        if (off) {                                    // shift by +1: need element h0 + VEC
            const int hx = (h0 + VEC >= Nh) ? 0 : h0 + VEC;
            const float x = __ldg(rowp + hx);
#pragma unroll
            for (int i = 0; i < VEC - 1; ++i) v[i] = v[i + 1];
            v[VEC - 1] = x;
        }
    } else if (D1 < 0) {
        if (!off) {                                   // shift by -1: need element h0 - 1
            const int hx = (h0 == 0) ? Nh - 1 : h0 - 1;
            const float x = __ldg(rowp + hx);
#pragma unroll
            for (int i = VEC - 1; i > 0; --i) v[i] = v[i - 1];
            v[0] = x;
        }
    }
#pragma unroll
    for (int i = 0; i < VEC; ++i) out[i] = ulm::to_fx(v[i]);
}

// Adds the two staples of the (MU, NU) plane to S for the VEC links of one thread (row a2):
//   S += e^{-i sigma+} + e^{-i sigma-},  -sigma+ = th_nu(x) + th_mu(x+nu) - th_nu(x+mu),
//                                        -sigma- = th_nu(x+mu-nu) + th_mu(x-nu) - th_nu(x-nu).
// tt/yy/zz hold the wrapped coordinates at displacement -1, 0, +1 in t, x2, x3.
template <int MU, int NU, int VEC>
__device__ __forceinline__ void staple_pair(const float* __restrict__ th, long long Vh, int Ns, int Nh, int p, int off,
                                            int h0, const int tt[3], const int yy[3], const int zz[3],
                                            float Sx[VEC], float Sy[VEC]) {
    constexpr int m0 = (MU == 0), m1 = (MU == 1), m2 = (MU == 2), m3 = (MU == 3);
    constexpr int n0 = (NU == 0), n1 = (NU == 1), n2 = (NU == 2), n3 = (NU == 3);
    auto rowptr = [&](int dir, int par, int d0, int d2, int d3) -> const float* {
        const long long row = ((long long)tt[d0 + 1] * Ns + zz[d3 + 1]) * Ns + yy[d2 + 1];
        return th + (long long)(dir * 2 + par) * Vh + row * Nh;
    };
    int A[VEC], B[VEC], C[VEC], D[VEC], E[VEC], F[VEC];
    load_row<VEC, 0>(rowptr(NU, p, 0, 0, 0), h0, off, Nh, A);                                   // theta_nu(x)
    load_row<VEC, n1>(rowptr(MU, 1 - p, n0, n2, n3), h0, off, Nh, B);                           // theta_mu(x+nu)
    load_row<VEC, m1>(rowptr(NU, 1 - p, m0, m2, m3), h0, off, Nh, C);                           // theta_nu(x+mu)
    load_row<VEC, m1 - n1>(rowptr(NU, p, m0 - n0, m2 - n2, m3 - n3), h0, off, Nh, D);           // theta_nu(x+mu-nu)
    load_row<VEC, -n1>(rowptr(MU, 1 - p, -n0, -n2, -n3), h0, off, Nh, E);                       // theta_mu(x-nu)
    load_row<VEC, -n1>(rowptr(NU, 1 - p, -n0, -n2, -n3), h0, off, Nh, F);                       // theta_nu(x-nu)
#pragma unroll
    for (int i = 0; i < VEC; ++i) {
        float c, s;
        ulm::sincos_fx<false>(A[i] + B[i] - C[i], c, s);
        Sx[i] += c; Sy[i] += s;
        ulm::sincos_fx<false>(D[i] + E[i] - F[i], c, s);
        Sx[i] += c; Sy[i] += s;
    }
}

// KIND 0 = heatbath, 1 = overrelaxation.  Block (Nh/VEC, BY, BZ); grid (Ns/BY, Ns/BZ, n_t)
// with n_t = Nt, or Nt*(d-1)/d active time layers for a masked spatial direction.
template <int KIND, int MU, int VEC>
__global__ void __launch_bounds__(256) k_update(const UpdateArgs P) {
    const int Ns = P.Ns, Nh = P.Nh, Nt = P.Nt;
    const int h0 = threadIdx.x * VEC;
    const int x2 = blockIdx.x * blockDim.y + threadIdx.y;
    const int x3 = blockIdx.y * blockDim.z + threadIdx.z;
    int t = blockIdx.z;
    if (MU != 0 && P.slab_d > 0) {                    // enumerate only the non-frozen layers
        const int dm = P.slab_d - 1;
        const int s = t / dm;
        t = s * P.slab_d + 1 + (t - s * dm);
    }
    const int p = P.parity;
    const int off = (p + x2 + x3 + t) & 1;            // x1 = 2h + off for the links of this thread

    // wrapped coordinates at displacement -1, 0, +1
    int tt[3], yy[3], zz[3];
    tt[1] = t;  tt[0] = (t == 0) ? Nt - 1 : t - 1;   tt[2] = (t == Nt - 1) ? 0 : t + 1;
    yy[1] = x2; yy[0] = (x2 == 0) ? Ns - 1 : x2 - 1; yy[2] = (x2 == Ns - 1) ? 0 : x2 + 1;
    zz[1] = x3; zz[0] = (x3 == 0) ? Ns - 1 : x3 - 1; zz[2] = (x3 == Ns - 1) ? 0 : x3 + 1;

    float Sx[VEC], Sy[VEC];
#pragma unroll
    for (int i = 0; i < VEC; ++i) { Sx[i] = 0.0f; Sy[i] = 0.0f; }

    staple_pair<MU, (MU + 1) & 3, VEC>(P.th, P.Vh, Ns, Nh, p, off, h0, tt, yy, zz, Sx, Sy);
    staple_pair<MU, (MU + 2) & 3, VEC>(P.th, P.Vh, Ns, Nh, p, off, h0, tt, yy, zz, Sx, Sy);
    staple_pair<MU, (MU + 3) & 3, VEC>(P.th, P.Vh, Ns, Nh, p, off, h0, tt, yy, zz, Sx, Sy);

    const long long row = ((long long)t * Ns + x3) * Ns + x2;
    float* own = P.th + (long long)(MU * 2 + p) * P.Vh + row * Nh + h0;
    float out[VEC];
    if (KIND == 1) {
        float old[VEC];
        if (VEC == 4) { const float4 q = *reinterpret_cast<const float4*>(own); old[0] = q.x; old[1 % VEC] = q.y; old[2 % VEC] = q.z; old[3 % VEC] = q.w; }
        else if (VEC == 2) { const float2 q = *reinterpret_cast<const float2*>(own); old[0] = q.x; old[1 % VEC] = q.y; }
        else old[0] = own[0];
#pragma unroll
        for (int i = 0; i < VEC; ++i) {
            const float alpha = ulm::atan2_acc(Sy[i], Sx[i]);
            out[i] = ulm::wrap(fmaf(2.0f, alpha, -old[i]));                  // overrelaxation (O2)
        }
    } else {
        const uint32_t site0 = (uint32_t)(row * Ns) + (uint32_t)(2 * h0 + off);   // canonical site index
        const uint32_t c3 = ((uint32_t)p << 2) | (uint32_t)MU;                    // tag 0 = heatbath
#pragma unroll
        for (int i = 0; i < VEC; ++i) {
            const float alpha = ulm::atan2_acc(Sy[i], Sx[i]);
            const float k = sqrtf(fmaf(Sx[i], Sx[i], Sy[i] * Sy[i]));
            const ulm::HbParams hp = ulm::hb_setup(P.beta * k);
            float phi = 0.0f;
            for (uint32_t n = 0; n < 64u; ++n) {                                  // cap 64 (O3)
                uint32_t w[4];
                ulm::philox4x32_10(site0 + 2u * i, P.sweep_lo, P.sweep_hi, (n << 8) | c3, P.key0, P.key1, w);
                if (ulm::hb_attempt(hp, w[0], w[1], w[2], phi)) break;
            }
            out[i] = ulm::wrap(alpha + phi);                                     // heatbath (O3)
        }
    }
    if (VEC == 4) *reinterpret_cast<float4*>(own) = make_float4(out[0], out[1 % VEC], out[2 % VEC], out[3 % VEC]);
    else if (VEC == 2) *reinterpret_cast<float2*>(own) = make_float2(out[0], out[1 % VEC]);
    else own[0] = out[0];
}

}  // namespace ulk
