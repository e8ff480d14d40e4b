// ul_persist.cuh -- one cooperative launch per compound sweep for lattices that live in L2 (the paper's 24^3 x Nt, P:92;
// BJ configs 1-4): the thread blocks stay resident, walk through the sub-steps of n_hb stochastic + n_or overrelaxation
// sweeps (S8(c)-O5: parity outer, direction inner) and meet at a grid barrier after each of them (the sub-steps are
// global barriers: same-colour links of different directions share plaquettes).  Same tiles, same device functions and
// same Philox counters as the one-launch-per-sub-step kernels of ul_update.cuh, so the links come out bit-identical;
// what goes away is the launch and drain per sub-step and the separate straggler and counter kernels.  Measured on B200: a
// grid barrier costs ~1.1 us at <= 200 blocks (3.2 us at 600) and a tile ~1.2-1.6 us of dependent latency, so the gain is
// 24^3 x 8: 147 -> 111 us per 1 + 3 compound sweep (heatbath sweep 66 -> 37 us); at 32^4 (1024 tiles) the graph-replayed
// launches are faster (280 against 350 us), so the host uses this kernel only up to PERSIST_MAX_TILES tiles.
//   * loads are L2-coherent (ld.global.cg): other blocks wrote the data earlier in the same launch;
//   * heatbath stragglers (both attempts of block 0 rejected) are finished by the SAME thread block from a
//     shared-memory queue right after its tile, so a heatbath sub-step needs one grid barrier, not two.
#pragma once
#include "ul_update.cuh"

namespace ulk {

struct PersistArgs {
    UpdateArgs u;              // lattice, beta, key, site offset, Metropolis width, sweep counter at the start (sweep_lo / sweep_hi)
    int n_hb, n_or;            // stochastic sweeps, then overrelaxation sweeps
    int stoch_kind;            // 0 heatbath, 2 Metropolis
    int gx, gy;                // tile grid of a time layer: x2 row pairs / blockDim.y, x3 / (blockDim.z / 2)
    int nt_time, nt_space;     // time layers a sub-step of direction 0 / of a spatial direction covers (masked: Nt (d-1)/d)
    unsigned* bar;             // grid barrier counters (grid_barrier below)
    unsigned bar_base;         // barriers passed by earlier launches of this context
};

constexpr int PERSIST_MAX_TILES = 256;
constexpr int PQ_CAP = 320;    // shared-memory straggler queue of a tile (<= 1024 links, 8-12 % pending; the rest is finished in place)

__device__ __forceinline__ unsigned ld_acquire_gpu(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// Grid barrier number k (k = 1, 2, ... counted over all launches of the context) of a cooperative, hence co-resident, grid:
// one release-arrival per block on a monotonic counter (fire and forget: no fence instruction, no returned value), then
// an acquire-poll until all gridDim.x blocks have arrived k times (wrapping 32-bit arithmetic, signed-difference compare).
// Measured and dropped: arrivals in groups of 16 on separate counters with a second level (slower: the round trips, not
// the serialisation of the atomics in L2, are what a barrier costs at <= 200 blocks).
__device__ __forceinline__ void grid_barrier(unsigned* bar, unsigned k, int tid) {
    __syncthreads();
    if (tid == 0) {
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");   // the block's stores (ordered by the bar.sync) before the arrival
        const unsigned target = k * gridDim.x;
        while ((int)(ld_acquire_gpu(bar) - target) < 0) {}
    }
    __syncthreads();
}

// The heatbath sub-step with the stragglers finished by the SAME thread block from a shared-memory queue (as in the persistent
// kernel below) instead of the striped global queue + k_hb_stragglers: for the small launches of a slab group (0.5-1 M links)
// a second launch costs more than the ~12 % of extra instructions.  Same counters and device functions: bit-identical links.
template <int MU, int VEC, bool DEVCTR>
__global__ void __launch_bounds__(256, UL_HB_MINB) k_update_hb_local(const UpdateArgs P) {
    __shared__ int4 sq[PQ_CAP];
    __shared__ int scount;
    const uint32_t sweep_lo = DEVCTR ? __ldg(P.sweep_dev) : P.sweep_lo, sweep_hi = DEVCTR ? __ldg(P.sweep_dev + 1) : P.sweep_hi;
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nthr = blockDim.x * blockDim.y * blockDim.z;
    if (tid == 0) scount = 0;
    __syncthreads();
    UpdateArgs Q = P;
    Q.queue = sq; Q.qcount = &scount; Q.qcap = PQ_CAP;            // tile index 0 -> sub-queue 0: the block's own queue
    update_tile<0, MU, VEC, false, true>(Q, blockIdx.x, blockIdx.y, blockIdx.z, gridDim.z, 0, sweep_lo, sweep_hi);
    __syncthreads();                                               // the tile's angles (placeholders for pending links) and its queue are written
    const int n = min(scount, PQ_CAP);
    int* own = P.th + (MU * 2 + P.parity) * P.Vh;
    const uint32_t c3 = ((uint32_t)P.parity << 2) | (uint32_t)MU;
    for (int e = tid; e < n; e += nthr) {
        const int4 q = sq[e];
        own[q.x] = ulm::hb_straggler(__int_as_float(q.z), __int_as_float(q.w), P.beta, (uint32_t)q.y, sweep_lo, sweep_hi, c3, P.key0, P.key1);
    }
}

template <int KIND, int VEC>
__device__ __forceinline__ void persist_tile(const UpdateArgs& P, int mu, int tx, int ty, int tz, int ntz, uint32_t sweep_lo, uint32_t sweep_hi) {
    switch (mu) {
        case 0: update_tile<KIND, 0, VEC, true, false>(P, tx, ty, tz, ntz, 0, sweep_lo, sweep_hi); break;
        case 1: update_tile<KIND, 1, VEC, true, false>(P, tx, ty, tz, ntz, 0, sweep_lo, sweep_hi); break;
        case 2: update_tile<KIND, 2, VEC, true, false>(P, tx, ty, tz, ntz, 0, sweep_lo, sweep_hi); break;
        default: update_tile<KIND, 3, VEC, true, false>(P, tx, ty, tz, ntz, 0, sweep_lo, sweep_hi); break;
    }
}

template <int VEC>
__global__ void __launch_bounds__(256) k_sweep_persistent(const PersistArgs A) {
    __shared__ int4 sq[PQ_CAP];
    __shared__ int scount;
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nthr = blockDim.x * blockDim.y * blockDim.z;
    UpdateArgs P = A.u;
    P.queue = sq; P.qcount = &scount; P.qcap = PQ_CAP;            // tile index 0 -> sub-queue 0: the block's own queue
    P.zflip = 0; P.z0 = 0;
    uint32_t sweep_lo = A.u.sweep_lo, sweep_hi = A.u.sweep_hi;
    unsigned kbar = A.bar_base;
    if (tid == 0) scount = 0;
    __syncthreads();
    for (int sw = 0; sw < A.n_hb + A.n_or; ++sw) {
        const int kind = sw < A.n_hb ? A.stoch_kind : 1;
        for (int parity = 0; parity < 2; ++parity) {
            P.parity = parity;
            for (int mu = 0; mu < 4; ++mu) {
                const int ntz = mu == 0 ? A.nt_time : A.nt_space;
                const int n_tiles = A.gx * A.gy * ntz;
                for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
                    const int tx = tile % A.gx, ty = (tile / A.gx) % A.gy, tz = tile / (A.gx * A.gy);
                    if (kind == 1) {
                        persist_tile<1, VEC>(P, mu, tx, ty, tz, ntz, sweep_lo, sweep_hi);
                    } else if (kind == 2) {
                        persist_tile<2, VEC>(P, mu, tx, ty, tz, ntz, sweep_lo, sweep_hi);
                    } else {
                        persist_tile<0, VEC>(P, mu, tx, ty, tz, ntz, sweep_lo, sweep_hi);
                        __syncthreads();                           // the tile's angles (placeholders for pending links) and its queue are written
                        const int n = min(scount, PQ_CAP);
                        int* own = P.th + (mu * 2 + parity) * P.Vh;
                        const uint32_t c3 = ((uint32_t)parity << 2) | (uint32_t)mu;
                        for (int e = tid; e < n; e += nthr) {
                            const int4 q = sq[e];
                            own[q.x] = ulm::hb_straggler(__int_as_float(q.z), __int_as_float(q.w), P.beta, (uint32_t)q.y, sweep_lo, sweep_hi, c3,
                                                         P.key0, P.key1);
                        }
                        __syncthreads();
                        if (tid == 0) scount = 0;
                        __syncthreads();
                    }
                }
                grid_barrier(A.bar, ++kbar, tid);
            }
        }
        if (kind != 1 && ++sweep_lo == 0u) ++sweep_hi;             // stochastic sweeps consume the counter (R19)
    }
}

}  // namespace ulk
