// ul_update.cuh -- link-update kernels: staple gather + heatbath / overrelaxation sub-step,
// full or slab-masked.
//
// Layout (row a1, BJ kernel 1): th[mu][par][row*Nh + h], fp32 angles in units of 2^-27 rad, where
//   row = (t*Ns + x3)*Ns + x2,  Nh = Ns/2,  par = (x1+x2+x3+t)&1,  x1 = 2h + ((par+x2+x3+t)&1).
// One sub-step (parity p, direction MU) updates the array th[MU][p] in place and reads the
// seven other arrays it depends on; it never reads an element another thread writes.
//
// Thread mapping: a thread owns VEC consecutive h of one row (VEC links).  Neighbours that are
// displaced in x2, x3, t keep the same h (aligned vector loads); a displacement in x1 shifts h
// by 0 or +-1 depending on the row's offset bit, which is handled with one extra scalar load.
// All addresses are 32-bit element offsets from the single base pointer (4V < 2^31 elements):
// own offset + periodic displacement deltas + uniform array offsets.
#pragma once
#include "ul_math.cuh"

namespace ulk {

struct UpdateArgs {
    float* th;            // internal layout, 8 arrays of Vh floats
    int Vh;               // V/2
    int Ns, Nh, Nt;
    int parity;           // sub-step parity p
    int slab_d;           // 0 = unmasked; else spatial links with t % slab_d == 0 are frozen
    float beta;
    uint32_t key0, key1;  // Philox key = seed
    uint32_t sweep_lo, sweep_hi;
};

// per-thread addressing state
struct Site {
    int e0;               // element offset of the thread's own chunk inside one array
    int dm[4], dp[4];     // element deltas for a displacement of -1 / +1 along t, (x1: 0), x2, x3
    int dxp, dxm;         // element deltas to the extra element of a +1 / -1 shifted chunk
    int off;              // x1 = 2h + off
};

// Loads, as fixed point, the VEC angles at element offset `idx` shifted by the x1-displacement D1
// (-1, 0, +1): x1 + 1 lives at h + off, x1 - 1 at h - 1 + off of the other-parity row.
template <int VEC, int D1>
__device__ __forceinline__ void load_row(const float* __restrict__ th, int idx, const Site& st, int out[VEC]) {
    float v[VEC];
    if (VEC == 4) {
        const float4 q = __ldg(reinterpret_cast<const float4*>(th + idx));
        v[0] = q.x; v[1 % VEC] = q.y; v[2 % VEC] = q.z; v[3 % VEC] = q.w;
    } else if (VEC == 2) {
        const float2 q = __ldg(reinterpret_cast<const float2*>(th + idx));
        v[0] = q.x; v[1 % VEC] = q.y;
    } else {
        v[0] = __ldg(th + idx);
    }
    if (D1 > 0) {
        if (st.off) {                                 // shift by +1: need element h0 + VEC
            const float x = __ldg(th + idx + st.dxp);
#pragma unroll
            for (int i = 0; i < VEC - 1; ++i) v[i] = v[i + 1];
            v[VEC - 1] = x;
        }
    } else if (D1 < 0) {
        if (!st.off) {                                // shift by -1: need element h0 - 1
            const float x = __ldg(th + idx + st.dxm);
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
template <int MU, int NU, int VEC>
__device__ __forceinline__ void staple_pair(const float* __restrict__ th, int Vh, int p, const Site& st,
                                            float Sx[VEC], float Sy[VEC]) {
    constexpr int m1 = (MU == 1), n1 = (NU == 1);
    const int a_nu_p = (NU * 2 + p) * Vh, a_nu_q = (NU * 2 + 1 - p) * Vh, a_mu_q = (MU * 2 + 1 - p) * Vh;
    int A[VEC], B[VEC], C[VEC], D[VEC], E[VEC], F[VEC];
    load_row<VEC, 0>(th, a_nu_p + st.e0, st, A);                                   // theta_nu(x)
    load_row<VEC, n1>(th, a_mu_q + st.e0 + st.dp[NU], st, B);                      // theta_mu(x+nu)
    load_row<VEC, m1>(th, a_nu_q + st.e0 + st.dp[MU], st, C);                      // theta_nu(x+mu)
    load_row<VEC, m1 - n1>(th, a_nu_p + st.e0 + st.dp[MU] + st.dm[NU], st, D);     // theta_nu(x+mu-nu)
    load_row<VEC, -n1>(th, a_mu_q + st.e0 + st.dm[NU], st, E);                     // theta_mu(x-nu)
    load_row<VEC, -n1>(th, a_nu_q + st.e0 + st.dm[NU], st, F);                     // theta_nu(x-nu)
#pragma unroll
    for (int i = 0; i < VEC; ++i) {
        ulm::cis_accumulate(A[i] + B[i] - C[i], Sx[i], Sy[i]);
        ulm::cis_accumulate(D[i] + E[i] - F[i], Sx[i], Sy[i]);
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
    const int sy = Nh, sz = Ns * Nh, stt = Ns * Ns * Nh;     // element strides of x2, x3, t
    Site st;
    st.off = (p + x2 + x3 + t) & 1;                   // x1 = 2h + off for the links of this thread
    st.e0 = ((t * Ns + x3) * Ns + x2) * Nh + h0;
    st.dp[0] = (t == Nt - 1) ? -(Nt - 1) * stt : stt;   st.dm[0] = (t == 0) ? (Nt - 1) * stt : -stt;
    st.dp[1] = 0;                                       st.dm[1] = 0;
    st.dp[2] = (x2 == Ns - 1) ? -(Ns - 1) * sy : sy;    st.dm[2] = (x2 == 0) ? (Ns - 1) * sy : -sy;
    st.dp[3] = (x3 == Ns - 1) ? -(Ns - 1) * sz : sz;    st.dm[3] = (x3 == 0) ? (Ns - 1) * sz : -sz;
    st.dxp = (h0 + VEC >= Nh) ? VEC - Nh : VEC;
    st.dxm = (h0 == 0) ? Nh - 1 : -1;

    float Sx[VEC], Sy[VEC];
#pragma unroll
    for (int i = 0; i < VEC; ++i) { Sx[i] = 0.0f; Sy[i] = 0.0f; }
    staple_pair<MU, (MU + 1) & 3, VEC>(P.th, P.Vh, p, st, Sx, Sy);
    staple_pair<MU, (MU + 2) & 3, VEC>(P.th, P.Vh, p, st, Sx, Sy);
    staple_pair<MU, (MU + 3) & 3, VEC>(P.th, P.Vh, p, st, Sx, Sy);

    float* own = P.th + ((MU * 2 + p) * P.Vh + st.e0);
    float out[VEC];
    if (KIND == 1) {
        float old[VEC];
        if (VEC == 4) { const float4 q = *reinterpret_cast<const float4*>(own); old[0] = q.x; old[1 % VEC] = q.y; old[2 % VEC] = q.z; old[3 % VEC] = q.w; }
        else if (VEC == 2) { const float2 q = *reinterpret_cast<const float2*>(own); old[0] = q.x; old[1 % VEC] = q.y; }
        else old[0] = own[0];
#pragma unroll
        for (int i = 0; i < VEC; ++i) {
            const float alpha = ulm::atan2_acc(Sy[i], Sx[i]);
            out[i] = ulm::to_units(ulm::wrap(fmaf(2.0f, alpha, -ulm::to_rad(old[i]))));   // overrelaxation (O2)
        }
    } else {
        const uint32_t site0 = (uint32_t)((st.e0 - h0) * 2 + 2 * h0 + st.off);            // canonical site index
        const uint32_t c3 = ((uint32_t)p << 2) | (uint32_t)MU;                            // tag 0 = heatbath
#pragma unroll
        for (int i = 0; i < VEC; ++i) {
            const float k = sqrtf(fmaf(Sx[i], Sx[i], Sy[i] * Sy[i]));
            const ulm::HbParams hp = ulm::hb_setup(P.beta * k);
            float sn = 0.0f, cs = 1.0f;
            uint32_t w[4];
            for (uint32_t n = 0; n < 64u; ++n) {                                          // cap 64 (O3)
                ulm::philox4x32_10(site0 + 2u * i, P.sweep_lo, P.sweep_hi, (n << 8) | c3, P.key0, P.key1, w);
                if (ulm::hb_attempt(hp, w[0], w[1], sn, cs)) break;
            }
            out[i] = ulm::to_units(ulm::hb_finish(Sx[i], Sy[i], sn, cs, (w[2] >> 31) != 0));   // heatbath (O3)
        }
    }
    if (VEC == 4) *reinterpret_cast<float4*>(own) = make_float4(out[0], out[1 % VEC], out[2 % VEC], out[3 % VEC]);
    else if (VEC == 2) *reinterpret_cast<float2*>(own) = make_float2(out[0], out[1 % VEC]);
    else own[0] = out[0];
}

}  // namespace ulk
