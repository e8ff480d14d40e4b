// ul_update_tma.cuh -- the overrelaxation sub-step with the neighbour rows STAGED IN SHARED MEMORY by bulk asynchronous
// copies (TMA engine: cp.async.bulk global -> shared, SASS UBLKCP, completion counted on an mbarrier): BJ north-star kernel (2)
// "staple gathering via shared-memory or TMA tile staging with halo", built as the A/B partner of the direct gather of
// ul_update.cuh (same tiles, same arithmetic through staple_pair_math / update_links, bit-identical links).
//
// A thread block of the direct kernel covers 2 blockDim.y consecutive x2 rows of one (x3, t): in every one of the eight
// link arrays that is ONE contiguous run of rows (128 bytes each at Ns = 64), and so is each of the 18 displaced row sets the
// staples need (a displacement in x3 or t moves the run, a displacement in x2 shifts it by one row, with the periodic
// boundary row as a second piece; a displacement in x1 stays inside the row).  One warp issues the 18 (+ boundary pieces)
// bulk copies, 72 KB per block at Ns = 64, all in flight at once; the threads then read their six angles per plane from
// shared memory instead of issuing 18 LDG.128 + the x1-shift scalars.  No reuse is gained (the DRAM traffic of the direct
// kernel is already the compulsory traffic: L1/L2 serve the stencil); what this variant tests is whether more bytes in
// flight per SM and fewer load instructions buy time.  Selected with UL_OR_TMA=1 (DESIGN.md section 5 has the measurement).
#pragma once
#include "ul_update.cuh"

namespace ulk {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}" ::"r"(
            smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src), "r"(bytes),
                 "r"(smem_u32(bar))
                 : "memory");
}

// the 4 angles at h0 .. h0+3 of a shared-memory row, shifted by the x1 displacement D1 as load_row does
template <int D1, int OFF>
__device__ __forceinline__ void load_row_s(const int* row, int h0, int Nh, int v[4]) {
    const int4 q = *reinterpret_cast<const int4*>(row + h0);
    v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
    if (D1 > 0) {
        if (OFF) {
            const int x = row[h0 + 4 >= Nh ? h0 + 4 - Nh : h0 + 4];
            v[0] = v[1]; v[1] = v[2]; v[2] = v[3]; v[3] = x;
        }
    } else if (D1 < 0) {
        if (!OFF) {
            const int x = row[h0 == 0 ? Nh - 1 : h0 - 1];
            v[3] = v[2]; v[2] = v[1]; v[1] = v[0]; v[0] = x;
        }
    }
}

// the two staples of plane (MU, NU) from the six staged row sets of that plane (set order A..F as in staple_pair)
template <int MU, int NU, int OFF>
__device__ __forceinline__ void staple_pair_s(const int* sets, int set_elems, int roff, int h0, int Nh, float Sx[4], float Sy[4]) {
    constexpr int m1 = (MU == 1), n1 = (NU == 1);
    int A[4], B[4], C[4], D[4], E[4], F[4];
    load_row_s<0, OFF>(sets + 0 * set_elems + roff, h0, Nh, A);              // theta_nu(x)
    load_row_s<n1, OFF>(sets + 1 * set_elems + roff, h0, Nh, B);             // theta_mu(x+nu)
    load_row_s<m1, OFF>(sets + 2 * set_elems + roff, h0, Nh, C);             // theta_nu(x+mu)
    load_row_s<m1 - n1, OFF>(sets + 3 * set_elems + roff, h0, Nh, D);        // theta_nu(x+mu-nu)
    load_row_s<-n1, OFF>(sets + 4 * set_elems + roff, h0, Nh, E);            // theta_mu(x-nu)
    load_row_s<-n1, OFF>(sets + 5 * set_elems + roff, h0, Nh, F);            // theta_nu(x-nu)
    staple_pair_math<4>(A, B, C, D, E, F, Sx, Sy);
}

// Block (Nh/4, BY, 2) as k_update with BZ = 1; grid (Ns/2/BY, Ns, n_t); dynamic shared memory 18 * 2 BY * Nh * 4 bytes.
template <int MU>
__global__ void __launch_bounds__(256, 3) k_update_or_tma(const UpdateArgs P) {
    extern __shared__ __align__(128) int tma_sm[];
    __shared__ __align__(8) unsigned long long mbar;
    const int Ns = P.Ns, Nh = P.Nh, Nt = P.Nt, p = P.parity;
    const int rows = 2 * blockDim.y, set_elems = rows * Nh;
    const int sel = threadIdx.z;
    const int x3 = blockIdx.y;
    int t = (P.zflip ? gridDim.z - 1 - blockIdx.z : blockIdx.z) + P.z0;
    if (MU != 0 && P.slab_d > 0) {                    // enumerate only the non-frozen layers
        const int dm = P.slab_d - 1;
        const int s = t / dm;
        t = s * P.slab_d + 1 + (t - s * dm);
    }
    const int x2lo = 2 * blockIdx.x * blockDim.y;
    const int x2 = x2lo + 2 * threadIdx.y + ((sel + p + x3 + t) & 1);
    const int h0 = threadIdx.x * 4;
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    if (tid == 0) {
        mbar_init(&mbar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    pdl_launch_dependents();
    pdl_wait();                                       // nothing is read before the previous launch is complete
    if (tid < 32) {
        if (tid == 0) mbar_arrive_expect_tx(&mbar, (uint32_t)(18 * set_elems * sizeof(int)));
        if (tid < 18) {
            const int n = tid / 6, which = tid - 6 * n;
            const int NU = (MU + 1 + n) & 3;
            // which: A theta_nu(x) | B theta_mu(x+nu) | C theta_nu(x+mu) | D theta_nu(x+mu-nu) | E theta_mu(x-nu) | F theta_nu(x-nu)
            const int dir = (which == 1 || which == 4) ? MU : NU;
            const int par = (which == 0 || which == 3) ? p : 1 - p;
            int d[4] = {0, 0, 0, 0};
            if (which == 1) d[NU] += 1;
            if (which == 2 || which == 3) d[MU] += 1;
            if (which >= 3) d[NU] -= 1;
            int tt = t + d[0], z3 = x3 + d[3];
            tt += tt < 0 ? Nt : (tt >= Nt ? -Nt : 0);
            z3 += z3 < 0 ? Ns : (z3 >= Ns ? -Ns : 0);
            const int* src = P.th + (size_t)(dir * 2 + par) * P.Vh + (size_t)(tt * Ns + z3) * Ns * Nh;   // row x2 = 0 of that (x3, t)
            int* dst = tma_sm + tid * set_elems;
            const int lo = x2lo + d[2];                                      // first row of the displaced run
            const uint32_t rowb = (uint32_t)(Nh * sizeof(int));
            if (lo < 0) {                                                    // periodic boundary: row Ns-1, then rows 0 .. rows-2
                bulk_g2s(dst, src + (size_t)(Ns - 1) * Nh, rowb, &mbar);
                bulk_g2s(dst + Nh, src, (uint32_t)(rows - 1) * rowb, &mbar);
            } else if (lo + rows > Ns) {                                     // rows lo .. Ns-1, then row 0
                bulk_g2s(dst, src + (size_t)lo * Nh, (uint32_t)(rows - 1) * rowb, &mbar);
                bulk_g2s(dst + (rows - 1) * Nh, src, rowb, &mbar);
            } else {
                bulk_g2s(dst, src + (size_t)lo * Nh, (uint32_t)rows * rowb, &mbar);
            }
        }
    }
    Site st;
    st.off = sel;
    st.e0 = ((t * Ns + x3) * Ns + x2) * Nh + h0;
    st.t = t;
    const int roff = (x2 - x2lo) * Nh;
    float Sx[4] = {0.0f, 0.0f, 0.0f, 0.0f}, Sy[4] = {0.0f, 0.0f, 0.0f, 0.0f};
    mbar_wait(&mbar, 0u);
    if (sel) {
        staple_pair_s<MU, (MU + 1) & 3, 1>(tma_sm + 0 * 6 * set_elems, set_elems, roff, h0, Nh, Sx, Sy);
        staple_pair_s<MU, (MU + 2) & 3, 1>(tma_sm + 1 * 6 * set_elems, set_elems, roff, h0, Nh, Sx, Sy);
        staple_pair_s<MU, (MU + 3) & 3, 1>(tma_sm + 2 * 6 * set_elems, set_elems, roff, h0, Nh, Sx, Sy);
    } else {
        staple_pair_s<MU, (MU + 1) & 3, 0>(tma_sm + 0 * 6 * set_elems, set_elems, roff, h0, Nh, Sx, Sy);
        staple_pair_s<MU, (MU + 2) & 3, 0>(tma_sm + 1 * 6 * set_elems, set_elems, roff, h0, Nh, Sx, Sy);
        staple_pair_s<MU, (MU + 3) & 3, 0>(tma_sm + 2 * 6 * set_elems, set_elems, roff, h0, Nh, Sx, Sy);
    }
    update_links<1, MU, 4, false>(P, st, h0, Sx, Sy, 0u, 0u, 0);
}

}  // namespace ulk
