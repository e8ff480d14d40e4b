// ul_update.cuh -- link-update kernels: staple gather + heatbath / overrelaxation sub-step,
// full or slab-masked.
//
// Layout (row a1, BJ kernel 1): th[mu][par][row*Nh + h], int32 binary angles (ul_math.cuh), where
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

#ifndef UL_PACKED_TRIG
#define UL_PACKED_TRIG 1   // staple trigonometry on pairs of links with FFMA2 / FMUL2
#endif

namespace ulk {

struct UpdateArgs {
    int* th;              // internal layout, 8 arrays of Vh binary angles
    int Vh;               // V/2
    int Ns, Nh, Nt;
    int parity;           // sub-step parity p
    int slab_d;           // 0 = unmasked; else spatial links with t % slab_d == 0 are frozen
    int z0;               // first time layer of the launch (blockIdx.z + z0; for a masked spatial direction in units of
                          // the enumerated non-frozen layers): launches restricted to a range of slabs
    int zflip;            // 1: the launch walks through its time layers from the last to the first (blocks are scheduled in
                          // grid order, so alternating the direction from sub-step to sub-step starts every sub-step on the
                          // layers the previous one left in L2; the result does not depend on the block order)
    float beta;
    uint32_t key0, key1;  // Philox key = seed
    uint32_t sweep_lo, sweep_hi;
    const uint32_t* sweep_dev;   // DEVCTR kernels (CUDA-graph replays) read the sweep counter from here instead
    int4* queue;          // heatbath stragglers: (element offset in th[mu][parity], site, Sx, Sy), see k_hb_stragglers
    int* qcount;          // [HB_NQ] entries in each sub-queue (zero before the launch) + [1] ticket of k_hb_stragglers
    int qcap;             // capacity of a sub-queue; sub-queue i = queue[i * qcap ...]
    // t-sharded full sweeps with peer-memory halo writes: the kernel stores the first / last halo_gl own time
    // layers it updates also into the neighbour shards' ghost layers (their link arrays, mapped peer memory over NVLink or
    // the same device), so no separate exchange step follows the sub-step.  Own layers: [halo_gl, halo_gl + halo_nt).
    int* peer_dn;         // link array of the shard below (t - 1 side), or nullptr
    int* peer_up;         // link array of the shard above
    int halo_gl, halo_nt;
    uint32_t site_offset; // added to the local canonical site index in the Philox counter (slab sharding: t0 * Ns^3)
    int met_delta_bt;     // Metropolis proposal half-width delta as a binary angle (0 < delta <= pi -> up to 2^31 - 1)
};

constexpr int HB_NQ = 64;      // the straggler queue is striped over HB_NQ compact sub-queues (thread block b appends to sub-queue b % HB_NQ)

// Programmatic dependent launch (sm_90+): with the launch attribute programmaticStreamSerialization a kernel's blocks are
// scheduled while the previous kernel of the stream drains; griddepcontrol.wait then blocks until that kernel has completed
// and its writes are visible.  Without the attribute both are no-ops.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// per-thread addressing state
struct Site {
    int e0;               // element offset of the thread's own chunk inside one array
    int dm[4], dp[4];     // element deltas for a displacement of -1 / +1 along t, (x1: 0), x2, x3
    int dxp, dxm;         // element deltas to the extra element of a +1 / -1 shifted chunk
    int off;              // x1 = 2h + off
    int t;                // local time layer
};

// Global loads of link angles.  COH = false: the read-only path (ld.global.nc), fine when the whole kernel only reads the
// arrays it does not write (one sub-step per launch).  COH = true: L2-coherent loads (ld.global.cg) for the persistent
// kernel, where other thread blocks wrote the data earlier in the same launch.
template <bool COH> __device__ __forceinline__ int4 ld4(const int* p) { return COH ? __ldcg(reinterpret_cast<const int4*>(p)) : __ldg(reinterpret_cast<const int4*>(p)); }
template <bool COH> __device__ __forceinline__ int2 ld2(const int* p) { return COH ? __ldcg(reinterpret_cast<const int2*>(p)) : __ldg(reinterpret_cast<const int2*>(p)); }
template <bool COH> __device__ __forceinline__ int ld1(const int* p) { return COH ? __ldcg(p) : __ldg(p); }

// Loads the VEC angles at element offset `idx` shifted by the x1-displacement D1 (-1, 0, +1):
// x1 + 1 lives at h + off, x1 - 1 at h - 1 + off of the other-parity row.
template <int VEC, int D1, int OFF, bool COH>
__device__ __forceinline__ void load_row(const int* __restrict__ th, int idx, const Site& st, int v[VEC]) {
    if (VEC == 4) {
        const int4 q = ld4<COH>(th + idx);
        v[0] = q.x; v[1 % VEC] = q.y; v[2 % VEC] = q.z; v[3 % VEC] = q.w;
    } else if (VEC == 2) {
        const int2 q = ld2<COH>(th + idx);
        v[0] = q.x; v[1 % VEC] = q.y;
    } else {
        v[0] = ld1<COH>(th + idx);
    }
    if (D1 > 0) {
        if (OFF) {                                    // shift by +1: need element h0 + VEC
            const int x = ld1<COH>(th + (idx + st.dxp));
#pragma unroll
            for (int i = 0; i < VEC - 1; ++i) v[i] = v[i + 1];
            v[VEC - 1] = x;
        }
    } else if (D1 < 0) {
        if (!OFF) {                                   // shift by -1: need element h0 - 1
            const int x = ld1<COH>(th + (idx + st.dxm));
#pragma unroll
            for (int i = VEC - 1; i > 0; --i) v[i] = v[i - 1];
            v[0] = x;
        }
    }
}

// S += e^{i(A+B-C)} + e^{i(D+E-F)} for the VEC links of one thread: the arithmetic of staple_pair, apart from where the six
// angles come from (global memory here, shared memory in ul_update_tma.cuh)
template <int VEC>
__device__ __forceinline__ void staple_pair_math(const int A[VEC], const int B[VEC], const int C[VEC], const int D[VEC], const int E[VEC],
                                                 const int F[VEC], float Sx[VEC], float Sy[VEC]) {
#if UL_POLY_TRIG && UL_PACKED_TRIG && !defined(UL_DBG_NOTRIG)
    if (VEC >= 2) {                                     // two links per FFMA2 / FMUL2 (bit-identical to the scalar form)
#pragma unroll
        for (int i = 0; i + 1 < VEC; i += 2) {
            ulm::f32x2 sx = ulm::pack2(Sx[i], Sx[i + 1]), sy = ulm::pack2(Sy[i], Sy[i + 1]);
            ulm::cis_pair_accumulate2((int)((unsigned)A[i] + (unsigned)B[i] - (unsigned)C[i]),
                                      (int)((unsigned)D[i] + (unsigned)E[i] - (unsigned)F[i]),
                                      (int)((unsigned)A[i + 1] + (unsigned)B[i + 1] - (unsigned)C[i + 1]),
                                      (int)((unsigned)D[i + 1] + (unsigned)E[i + 1] - (unsigned)F[i + 1]), sx, sy);
            ulm::unpack2(sx, Sx[i], Sx[i + 1]);
            ulm::unpack2(sy, Sy[i], Sy[i + 1]);
        }
        return;
    }
#endif
#pragma unroll
    for (int i = 0; i < VEC; ++i) {
        ulm::cis_pair_accumulate((int)((unsigned)A[i] + (unsigned)B[i] - (unsigned)C[i]),
                                 (int)((unsigned)D[i] + (unsigned)E[i] - (unsigned)F[i]), Sx[i], Sy[i]);
    }
}

// Adds the two staples of the (MU, NU) plane to S for the VEC links of one thread (row a2):
//   S += e^{-i sigma+} + e^{-i sigma-},  -sigma+ = th_nu(x) + th_mu(x+nu) - th_nu(x+mu),
//                                        -sigma- = th_nu(x+mu-nu) + th_mu(x-nu) - th_nu(x-nu).
// The phase sums are wrapping int32 adds: exact and already reduced mod 2 pi.
template <int MU, int NU, int VEC, int OFF, bool COH>
__device__ __forceinline__ void staple_pair(const int* __restrict__ th, int Vh, int p, const Site& st,
                                            float Sx[VEC], float Sy[VEC]) {
    constexpr int m1 = (MU == 1), n1 = (NU == 1);
    const int a_nu_p = (NU * 2 + p) * Vh, a_nu_q = (NU * 2 + 1 - p) * Vh, a_mu_q = (MU * 2 + 1 - p) * Vh;
    int A[VEC], B[VEC], C[VEC], D[VEC], E[VEC], F[VEC];
    load_row<VEC, 0, OFF, COH>(th, a_nu_p + st.e0, st, A);                                   // theta_nu(x)
    load_row<VEC, n1, OFF, COH>(th, a_mu_q + st.e0 + st.dp[NU], st, B);                      // theta_mu(x+nu)
    load_row<VEC, m1, OFF, COH>(th, a_nu_q + st.e0 + st.dp[MU], st, C);                      // theta_nu(x+mu)
    load_row<VEC, m1 - n1, OFF, COH>(th, a_nu_p + st.e0 + st.dp[MU] + st.dm[NU], st, D);     // theta_nu(x+mu-nu)
    load_row<VEC, -n1, OFF, COH>(th, a_mu_q + st.e0 + st.dm[NU], st, E);                     // theta_mu(x-nu)
    load_row<VEC, -n1, OFF, COH>(th, a_nu_q + st.e0 + st.dm[NU], st, F);                     // theta_nu(x-nu)
    staple_pair_math<VEC>(A, B, C, D, E, F, Sx, Sy);
}

template <typename T, int VEC>
__device__ __forceinline__ T pick(const T v[VEC], int j) {        // v[j] without dynamic register indexing
    T r = v[0];
#pragma unroll
    for (int i = 1; i < VEC; ++i) r = (j == i) ? v[i] : r;
    return r;
}

// The staple sums of the VEC links of one thread, compiled separately for the two values of the row's
// offset bit OFF (x1 = 2h + OFF) so that the x1-shifted neighbour rows are selected by register naming at
// compile time instead of predicated moves.
template <int MU, int VEC, int OFF, bool COH>
__device__ __forceinline__ void gather_staples(const UpdateArgs& P, const Site& st, float Sx[VEC], float Sy[VEC]) {
#pragma unroll
    for (int i = 0; i < VEC; ++i) { Sx[i] = 0.0f; Sy[i] = 0.0f; }
    staple_pair<MU, (MU + 1) & 3, VEC, OFF, COH>(P.th, P.Vh, P.parity, st, Sx, Sy);
    staple_pair<MU, (MU + 2) & 3, VEC, OFF, COH>(P.th, P.Vh, P.parity, st, Sx, Sy);
    staple_pair<MU, (MU + 3) & 3, VEC, OFF, COH>(P.th, P.Vh, P.parity, st, Sx, Sy);
}

// The update proper from the staple sums.  KIND 0 = heatbath, 1 = overrelaxation.
template <int KIND, int MU, int VEC, bool COH>
__device__ __forceinline__ void update_links(const UpdateArgs& P, const Site& st, const int h0, float Sx[VEC], float Sy[VEC],
                                             const uint32_t sweep_lo, const uint32_t sweep_hi, const int blk) {
    const int p = P.parity;
    int* own = P.th + ((MU * 2 + p) * P.Vh + st.e0);
    int out[VEC];
    if (KIND == 1) {
        int old[VEC];
        if (VEC == 4) { const int4 q = COH ? __ldcg(reinterpret_cast<const int4*>(own)) : *reinterpret_cast<const int4*>(own); old[0] = q.x; old[1 % VEC] = q.y; old[2 % VEC] = q.z; old[3 % VEC] = q.w; }
        else if (VEC == 2) { const int2 q = COH ? __ldcg(reinterpret_cast<const int2*>(own)) : *reinterpret_cast<const int2*>(own); old[0] = q.x; old[1 % VEC] = q.y; }
        else old[0] = COH ? __ldcg(own) : own[0];
#pragma unroll
        for (int i = 0; i < VEC; i += 2) {            // overrelaxation (O2): theta' = 2 alpha - theta, exact mod 2 pi
            int al[2];
            if (i + 1 < VEC) ulm::atan2_bt2(Sy[i], Sx[i], Sy[(i + 1) % VEC], Sx[(i + 1) % VEC], al[0], al[1]);   // two links per FFMA2
            else al[0] = ulm::atan2_bt(Sy[i], Sx[i]);
#pragma unroll
            for (int j = 0; j < 2 && i + j < VEC; ++j)
                out[(i + j) % VEC] = (int)(2u * (unsigned)al[j] - (unsigned)old[(i + j) % VEC]);
        }
    } else if (KIND == 2) {
        // Metropolis (DESIGN R21): one hit, theta' = theta + delta (2 u1 - 1), accept iff
        // u2 <= exp(beta k [cos(theta' - alpha) - cos(theta - alpha)]).  With d = theta' - theta (an exact integer
        // number of binary-angle units: v delta 2^-23, v = 2^24 u1 - 2^23 odd) the exponent is, without alpha and
        // without cancellation,  beta 2 sin(d/2) [Sy cos(theta + d/2) - Sx sin(theta + d/2)].
        int old[VEC];
        if (VEC == 4) { const int4 q = COH ? __ldcg(reinterpret_cast<const int4*>(own)) : *reinterpret_cast<const int4*>(own); old[0] = q.x; old[1 % VEC] = q.y; old[2 % VEC] = q.z; old[3 % VEC] = q.w; }
        else if (VEC == 2) { const int2 q = COH ? __ldcg(reinterpret_cast<const int2*>(own)) : *reinterpret_cast<const int2*>(own); old[0] = q.x; old[1 % VEC] = q.y; }
        else old[0] = COH ? __ldcg(own) : own[0];
        const uint32_t site0 = (uint32_t)((st.e0 - h0) * 2 + 2 * h0 + st.off) + P.site_offset;            // canonical site index
        const uint32_t c3 = (3u << 3) | ((uint32_t)p << 2) | (uint32_t)MU;                // tag 3 = Metropolis, attempt 0
#pragma unroll
        for (int i = 0; i < VEC; ++i) {
            uint32_t w[4];
            ulm::philox4x32_10(site0 + 2u * i, sweep_lo, sweep_hi, c3, P.key0, P.key1, w);
            const int v = (int)((w[0] >> 8) | 1u) - (1 << 23);                            // (2 u1 - 1) 2^23, odd, |v| < 2^23
            const int d = (int)(((long long)v * (long long)P.met_delta_bt) >> 23);        // |d| <= pi
            const int h = d >> 1;                                                         // |h| <= pi/2: no reduction needed
            const float rh = __int2float_rn(h) * ulm::BT_TO_RAD;
            const float zh = rh * rh;
            float sh = fmaf(2.598120545371785e-06f, zh, -0.00019805740157607943f);        // sin(d/2), degree 9 on |r| <= pi/2
            sh = fmaf(sh, zh, 0.008333005011081696f);
            sh = fmaf(sh, zh, -0.16666656732559204f);
            sh = fmaf(sh, zh * rh, rh);
            float cm = 0.0f, sm = 0.0f;
            ulm::cis_accumulate((int)((unsigned)old[i] + (unsigned)h), cm, sm);           // cos, sin of theta + d/2
            const float gain = P.beta * 2.0f * sh * fmaf(Sy[i], cm, -(Sx[i] * sm));
            const bool accept = ulm::u01(w[1]) <= ulm::mufu_ex2(gain * 1.44269504088896340736f);
            out[i] = accept ? (int)((unsigned)old[i] + (unsigned)d) : old[i];
        }
    } else {
        // Heatbath (O3).  Attempt n of a link is a pure function of (site, sweep, n): Philox block n >> 1, word pair
        // n & 1 (DESIGN R19).  Every link gets its block 0, i.e. attempts 0 and 1, here with the warp converged: the two
        // attempts of a link are the two lanes of the packed arithmetic, and the first accepted one is taken.  The links
        // that rejected both (8-12 %) go to this block's segment of the straggler queue and k_hb_stragglers finishes them
        // from block 1 on (same counters, same device functions), so no warp loops for its unluckiest lane.
        const uint32_t site0 = (uint32_t)((st.e0 - h0) * 2 + 2 * h0 + st.off) + P.site_offset;            // canonical site index
        const uint32_t c3 = ((uint32_t)p << 2) | (uint32_t)MU;                            // tag 0 = heatbath, block 0
        // A pair of links is taken all the way to its new angles before the next pair starts (short live ranges: 64
        // registers); the angle written for a link that is still pending is a placeholder that k_hb_stragglers overwrites.
        uint32_t pend = 0u, zero = 0u;
        float a[VEC];
#pragma unroll
        for (int i = 0; i < VEC; ++i) {
            const float k2 = fmaf(Sx[i], Sx[i], Sy[i] * Sy[i]);
            if (k2 == 0.0f) { Sx[i] = 1.0f; Sy[i] = 0.0f; zero |= 1u << i; }               // k = 0: alpha = 0 (O1)
            a[i] = P.beta * ulm::mufu_sqrt(k2);
        }
#pragma unroll
        for (int i = 0; i < VEC; i += 2) {
            ulm::HbParams hp[2];
            if (i + 1 < VEC) ulm::hb_setup2(a[i], a[(i + 1) % VEC], hp[0], hp[1]);        // the per-link constants on pairs of links
            else hp[0] = ulm::hb_setup(a[i]);
            float sn[2], cs[2];
            bool ng[2] = {false, false};
#pragma unroll
            for (int j = 0; j < 2 && i + j < VEC; ++j) {
                uint32_t w[4];
                ulm::philox4x32_10(site0 + 2u * (i + j), sweep_lo, sweep_hi, c3, P.key0, P.key1, w);
                bool acc;
                ulm::hb_block(hp[j], w, sn[j], cs[j], acc, ng[j]);
                pend |= (acc ? 0u : 1u) << (i + j);
            }
            if (i + 1 < VEC)
                ulm::hb_finish2(ulm::pack2(Sx[i], Sx[(i + 1) % VEC]), ulm::pack2(Sy[i], Sy[(i + 1) % VEC]), ulm::pack2(sn[0], sn[1]),
                                ulm::pack2(cs[0], cs[1]), ng[0], ng[1], out[i], out[(i + 1) % VEC]);
            else
                out[i] = ulm::hb_finish(Sx[i], Sy[i], sn[0], cs[0], ng[0]);
        }
        // the lanes of this warp that exist: every thread of the block reaches this point (no early exits), so the mask
        // is known from the block size
        const int tid_ = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
        const int in_warp = min(32, (int)(blockDim.x * blockDim.y * blockDim.z) - (tid_ & ~31));
        const unsigned wmask = in_warp == 32 ? 0xffffffffu : ((1u << in_warp) - 1u);
        if (__ballot_sync(wmask, pend != 0u)) {                                           // warp-uniform
            const unsigned lt = (1u << (tid_ & 31)) - 1u;
            int off[VEC], total = 0;
#pragma unroll
            for (int i = 0; i < VEC; ++i) {                                               // slots: link index major, lane minor
                const unsigned b = __ballot_sync(wmask, ((pend >> i) & 1u) != 0u);
                off[i] = total + __popc(b & lt);
                total += __popc(b);
            }
            int base = 0;
            const int qi = blk & (HB_NQ - 1);
            if ((tid_ & 31) == 0) base = atomicAdd(P.qcount + qi, total);                 // one atomic per warp, spread over HB_NQ counters
            base = __shfl_sync(wmask, base, 0);
#pragma unroll
            for (int i = 0; i < VEC; ++i)
                if ((pend >> i) & 1u) {
                    const int pos = base + off[i];
                    const float sx = ((zero >> i) & 1u) ? 0.0f : Sx[i];
                    if (pos < P.qcap)
                        P.queue[(size_t)qi * P.qcap + pos] = make_int4(st.e0 + i, (int)(site0 + 2u * i), __float_as_int(sx), __float_as_int(Sy[i]));
                    else                                                                  // sub-queue full (never seen): finish here
                        out[i] = ulm::hb_straggler_call(sx, Sy[i], P.beta, site0 + 2u * i, sweep_lo, sweep_hi, c3, P.key0, P.key1);
                }
        }
    }
    auto store = [&](int* dst) {
        if (VEC == 4) *reinterpret_cast<int4*>(dst) = make_int4(out[0], out[1 % VEC], out[2 % VEC], out[3 % VEC]);
        else if (VEC == 2) *reinterpret_cast<int2*>(dst) = make_int2(out[0], out[1 % VEC]);
        else dst[0] = out[0];
    };
    store(own);
    if (P.peer_dn != nullptr) {                                   // (uniform) boundary layers also go to the neighbours' ghost layers
        const int arr = (MU * 2 + p) * P.Vh + st.e0, shift = P.halo_nt * (P.Ns * P.Ns * P.Nh);
        if (st.t < 2 * P.halo_gl) store(P.peer_dn + arr + shift);                // first own layers -> upper ghost of the shard below
        if (st.t >= P.halo_nt) store(P.peer_up + arr - shift);                   // last own layers -> lower ghost of the shard above
    }
}


__global__ void k_bump_sweep(uint32_t* sweep) {                 // ++counter (64 bit) at the end of a stochastic sweep of a graph
    const uint32_t lo = sweep[0] + 1u;
    sweep[0] = lo;
    if (lo == 0u) sweep[1] += 1u;
}
__global__ void k_set_sweep(uint32_t* sweep, uint32_t lo, uint32_t hi) { sweep[0] = lo; sweep[1] = hi; }

// Block (Nh/VEC, BYH, 2 BZ); grid (Ns/2/BYH, Ns/BZ, n_t) with n_t = Nt, or Nt*(d-1)/d active time layers for
// a masked spatial direction.  The x2 rows are taken in pairs (2j, 2j+1): threads with threadIdx.z < BZ
// take the row of the pair whose offset bit is 0, the others the row whose offset bit is 1, so the offset
// bit is uniform over a warp whenever (Nh/VEC) BYH BZ is a multiple of 32 (any Ns that is a multiple of
// 16; smaller lattices still compute the same thing, with both branches issued).
#ifndef UL_HB_MINB
#define UL_HB_MINB 4
#endif
#ifndef UL_ORG_MINB
#define UL_ORG_MINB 4   // graph-replayed overrelaxation launches (small lattices, slab groups out of L2): 64 registers, 4 blocks per SM (with the
                        // shorter instruction sequence of the gather 1-5 % faster than 3 blocks of up to 80 registers: bench step 49.9 -> 49.2 ms)
#endif
#ifndef UL_OR_MINB
#define UL_OR_MINB 4   // overrelaxation / Metropolis launches over the whole lattice (HBM-bound): 64 registers, 4 blocks per SM.  With the
#endif                 // shorter instruction sequence of the gather this is the optimum again (OR sweep on 64^4: 3 blocks 429 us, 4 blocks
                       // 406 us, 5 blocks of 48 registers 418 us, 6 blocks spill; before the cuts 5 blocks won, 440 -> 417 us)
// One tile (= one thread block's worth) of a sub-step: tile coordinates (tx, ty, tz) of a (gx, gy, ntz) tile grid, blk = the
// tile's linear index (picks the straggler sub-queue).
template <int KIND, int MU, int VEC, bool COH, bool PDL>
__device__ __forceinline__ void update_tile(const UpdateArgs& P, const int tx, const int ty, const int tz, const int ntz, const int blk,
                                            const uint32_t sweep_lo, const uint32_t sweep_hi) {
    const int Ns = P.Ns, Nh = P.Nh, Nt = P.Nt;
    const int h0 = threadIdx.x * VEC;
    const int bz = blockDim.z >> 1;
    const int sel = threadIdx.z >= bz ? 1 : 0;
    const int x3 = ty * bz + (threadIdx.z - sel * bz);
    int t = (P.zflip ? ntz - 1 - tz : tz) + P.z0;
    if (MU != 0 && P.slab_d > 0) {                    // enumerate only the non-frozen layers
        const int dm = P.slab_d - 1;
        // s = t / dm without the ~25 instructions of an integer division in every thread: nothing to do at thickness 2;
        // otherwise the truncated float quotient of t + 1/2, exact for t < 2^20 (the fractional part of (t + 1/2) / dm is
        // at least 1 / (2 dm) away from an integer, the approximate quotient is off by < 2^-21 (t / dm)); beyond that
        // (no lattice that fits a GPU has 2^20 time layers) the division
        const int s = dm == 1 ? t : (t < (1 << 20) ? __float2int_rz(__fdividef(__int2float_rn(t) + 0.5f, __int2float_rn(dm))) : t / dm);
        t = s * P.slab_d + 1 + (t - s * dm);
    }
    const int p = P.parity;
    const int x2 = 2 * (tx * blockDim.y + threadIdx.y) + ((sel + p + x3 + t) & 1);
    const int sy = Nh, sz = Ns * Nh, stt = Ns * Ns * Nh;     // element strides of x2, x3, t
    Site st;
    st.off = sel;                                     // = (p + x2 + x3 + t) & 1: x1 = 2h + off for the links of this thread
    st.e0 = ((t * Ns + x3) * Ns + x2) * Nh + h0;
    st.t = t;
    st.dp[0] = (t == Nt - 1) ? -(Nt - 1) * stt : stt;   st.dm[0] = (t == 0) ? (Nt - 1) * stt : -stt;
    st.dp[1] = 0;                                       st.dm[1] = 0;
    st.dp[2] = (x2 == Ns - 1) ? -(Ns - 1) * sy : sy;    st.dm[2] = (x2 == 0) ? (Ns - 1) * sy : -sy;
    st.dp[3] = (x3 == Ns - 1) ? -(Ns - 1) * sz : sz;    st.dm[3] = (x3 == 0) ? (Ns - 1) * sz : -sz;
    st.dxp = (h0 + VEC >= Nh) ? VEC - Nh : VEC;
    st.dxm = (h0 == 0) ? Nh - 1 : -1;
    if (PDL) {
        pdl_launch_dependents();                      // the next launch of the stream may start its own index arithmetic
        pdl_wait();                                   // ... but nothing is read or written before the previous launch is complete
    }
    float Sx[VEC], Sy[VEC];
    if (KIND != 0) {
        // overrelaxation, Metropolis: the short tail is compiled into both branches (56 registers, 4 blocks per SM)
        if (sel) { gather_staples<MU, VEC, 1, COH>(P, st, Sx, Sy); update_links<KIND, MU, VEC, COH>(P, st, h0, Sx, Sy, sweep_lo, sweep_hi, blk); }
        else { gather_staples<MU, VEC, 0, COH>(P, st, Sx, Sy); update_links<KIND, MU, VEC, COH>(P, st, h0, Sx, Sy, sweep_lo, sweep_hi, blk); }
    } else {
        // heatbath: one copy of the sampler after the branch keeps it at 64 registers (4 blocks per SM)
        if (sel) gather_staples<MU, VEC, 1, COH>(P, st, Sx, Sy);
        else gather_staples<MU, VEC, 0, COH>(P, st, Sx, Sy);
        update_links<KIND, MU, VEC, COH>(P, st, h0, Sx, Sy, sweep_lo, sweep_hi, blk);
    }
}

template <int KIND, int MU, int VEC, bool DEVCTR>
__global__ void __launch_bounds__(256, KIND == 0 ? UL_HB_MINB : (DEVCTR ? UL_ORG_MINB : UL_OR_MINB)) k_update(const UpdateArgs P) {
    // the sweep counter: a kernel argument (uniform registers), or, for launches replayed from a CUDA graph, device memory
    const uint32_t sweep_lo = DEVCTR ? __ldg(P.sweep_dev) : P.sweep_lo, sweep_hi = DEVCTR ? __ldg(P.sweep_dev + 1) : P.sweep_hi;
    update_tile<KIND, MU, VEC, false, true>(P, blockIdx.x, blockIdx.y, blockIdx.z, gridDim.z, blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z),
                                            sweep_lo, sweep_hi);
}

// Finishes the heatbath links that k_update<0,...> queued: blocks 1, 2, ... of their Philox streams with the same
// counters and the same device functions as the main kernel (so the result does not depend on where a link is finished),
// until accept or the cap of 64 attempts (O3).  Grid (HB_NQ, QB): the QB thread blocks of a sub-queue stride over its
// entries, one entry per thread and step (no shared memory, no barrier: the grid is one wave and every lane has work).
// The last block to finish zeroes the counters for the next heatbath sub-step.
#ifndef UL_HBS_MINB
#define UL_HBS_MINB 4
#endif
template <bool DEVCTR>
__global__ void __launch_bounds__(256, UL_HBS_MINB) k_hb_stragglers(const UpdateArgs P, int mu) {
    const uint32_t c3 = ((uint32_t)P.parity << 2) | (uint32_t)mu;
    const uint32_t sweep_lo = DEVCTR ? __ldg(P.sweep_dev) : P.sweep_lo, sweep_hi = DEVCTR ? __ldg(P.sweep_dev + 1) : P.sweep_hi;
    pdl_launch_dependents();
    pdl_wait();
    const int n = min(P.qcount[blockIdx.x], P.qcap);                                      // a count above qcap: the rest was finished in place
    const int4* q0 = P.queue + (size_t)blockIdx.x * P.qcap;
    int* own = P.th + (mu * 2 + P.parity) * P.Vh;
    for (int e = blockIdx.y * blockDim.x + threadIdx.x; e < n; e += gridDim.y * blockDim.x) {
        const int4 q = q0[e];
        // q.y = the site index, all 32 bits (ghost-layer sites of a shard wrap); (q.z, q.w) = the staple sum, (0, 0) if k = 0
        const int v = ulm::hb_straggler(__int_as_float(q.z), __int_as_float(q.w), P.beta, (uint32_t)q.y, sweep_lo, sweep_hi, c3, P.key0, P.key1);
        own[q.x] = v;
        if (P.peer_dn != nullptr) {                                                       // as in update_links
            const int stt = P.Ns * P.Ns * P.Nh, t = q.x / stt, arr = (mu * 2 + P.parity) * P.Vh + q.x;
            if (t < 2 * P.halo_gl) P.peer_dn[arr + P.halo_nt * stt] = v;
            if (t >= P.halo_nt) P.peer_up[arr - P.halo_nt * stt] = v;
        }
    }
    __syncthreads();                                                                      // every thread of the block has read its count
    if (threadIdx.x == 0) {
        const int nblk = gridDim.x * gridDim.y;
        if (atomicAdd(P.qcount + HB_NQ, 1) == nblk - 1) {                                 // the last block: nobody reads the counts any more
#pragma unroll 1
            for (int i = 0; i <= HB_NQ; ++i) P.qcount[i] = 0;
        }
    }
}

}  // namespace ulk
