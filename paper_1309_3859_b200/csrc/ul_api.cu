// ul_api.cu -- host driver and C ABI of libul.so (include/ul.h).
//
// The host only enqueues kernels: the sweep schedule (S8(c)-O5), the sub-update recipe
// and the nesting of Algorithm 1.  Every arithmetic step of the hot
// path runs in the kernels of ul_update.cuh / ul_measure.cuh.  There is no CPU fallback.
#include "../../include/ul.h"

#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "ul_measure.cuh"
#include "ul_update.cuh"
#include "ul_persist.cuh"
#include "ul_update_tma.cuh"

namespace {

// NVTX ranges around the host-side steps (visible in nsys / ncu --nvtx; a no-op without a tool attached)
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

// the entry points run on the context's device, whatever the caller's current device is
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const ul_ctx* c);
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

constexpr int NBLK = 592;   // blocks of the two-stage reductions: 4 per SM on 148 SMs
constexpr int TBLK = 8 * NBLK;   // blocks of the slab-table kernel (grid-stride; one partial per block and column)

constexpr int KBATCH = 8;   // configurations accumulated per read-modify-write pass over the accumulators

struct Workspace {           // byte offsets into the measurement workspace
    size_t U = 0, Um = 0, Ot = 0, fps = 0, A2 = 0, B2 = 0, A4 = 0, B4 = 0, partial = 0, result = 0, total = 0;
    int kb = 1;              // batch depth: slots of U (and of Ot when field points are measured)
};

size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

// blocks per (r, field point) of k_replay_reduce: >= 16 sites per thread and direction, so that the 24-value block
// reduction is amortised
int replay_blocks(long long n_slab_sites) {
    const long long nb = n_slab_sites / (256 * 16);
    return nb < 1 ? 1 : (nb > NBLK ? NBLK : (int)nb);
}

Workspace plan_workspace(int Ns, int Nt, int d_in, int d_out, int r_max, int n_fp, bool replay = false, bool multihit = false) {
    Workspace w;
    const size_t Vs = (size_t)Ns * Ns * Ns;
    const size_t n_in = (size_t)(Nt / d_in), n_out = d_out > 0 ? (size_t)(Nt / d_out) : 0;
    const size_t F12 = (size_t)n_fp * 12, R = (size_t)r_max;
    const size_t FB = replay ? 1 : F12;          // replay: the B2 slot holds the weights W (one A-sized array), no TO sums
    const size_t ot_slots = replay ? 1 : 0;      // replay: one Ot table (pass 2 is not batched); else kb slots
    // batch depth: KBATCH, reduced if the per-configuration tables would outgrow the accumulators they feed
    const size_t table = n_in * Vs * (16 + (n_fp > 0 && !replay ? 48 : 0));
    const size_t accum = 3 * R * n_in * Vs * 16 * (1 + FB);
    int kb = KBATCH;
    while (kb > 1 && (size_t)kb * table > accum / 2 + ((size_t)64 << 20)) kb >>= 1;
    w.kb = kb;
    size_t o = 0;
    w.U = o;   o = align_up(o + (size_t)kb * n_in * Vs * 16);
    w.Um = o;  o = align_up(o + (multihit ? (size_t)kb * n_in * Vs * 16 : 0));
    w.Ot = o;  o = align_up(o + (n_fp > 0 ? (ot_slots ? ot_slots : (size_t)kb) * 12 * n_in * Vs * sizeof(float) : 0));
    w.fps = o; o = align_up(o + (size_t)(n_fp > 0 ? n_fp : 1) * 3 * sizeof(int));
    w.A2 = o;  o = align_up(o + 3 * R * n_in * Vs * 16);
    w.B2 = o;  o = align_up(o + 3 * R * n_in * FB * Vs * 16);
    w.A4 = o;  o = align_up(o + 3 * R * n_out * Vs * 16);
    w.B4 = o;  o = align_up(o + 3 * R * n_out * FB * Vs * 16);
    const size_t n_entries = R * (1 + F12);
    size_t np = 2 * n_entries;
    if (np < 12 * (TBLK / NBLK)) np = 12 * (TBLK / NBLK);
    size_t partial_doubles = np * NBLK;
    if (replay) {                                   // fields: replay_blocks() partials per entry; correlators: NBLK per entry
        const size_t nb = replay_blocks((long long)(n_in * Vs));
        partial_doubles = 2 * R * NBLK + 2 * R * F12 * nb;
        if (partial_doubles < (size_t)12 * TBLK) partial_doubles = (size_t)12 * TBLK;
    }
    w.partial = o; o = align_up(o + partial_doubles * sizeof(double));
    w.result = o;  o = align_up(o + (2 * n_entries + 12 + 12) * sizeof(double));   // corr|field, vacuum, column sums
    w.total = o;
    return w;
}

}  // namespace

struct GraphKey {
    int n_hb, n_or, slab_d, alg;
    double beta, met_delta;
    uint32_t site_offset;
    bool operator==(const GraphKey& o) const {
        return n_hb == o.n_hb && n_or == o.n_or && slab_d == o.slab_d && alg == o.alg &&
               beta == o.beta && met_delta == o.met_delta && site_offset == o.site_offset;
    }
};
// one compound sub-update of a ROUND of slab groups (S groups side by side, each on its own stream), captured as one graph
struct RoundGraph {
    int g0, grp, S, n_hb, n_or, sub_k, slab_d, alg;
    int n_sub, kb, r_max, n_fp, multihit;   // the whole round: n_sub x (sub-update of the S groups, tables) + accumulation passes
    const void* work; size_t ws_total;     // the workspace the table and accumulation launches were captured with
    double beta, met_delta;
    uint32_t site_offset;
    cudaGraphExec_t exec = nullptr;
    uint64_t launches = 0;
};
struct CachedGraph {
    GraphKey key;
    cudaGraphExec_t exec = nullptr;
    uint64_t launches = 0;
};

struct ul_ctx {
    int Ns = 0, Nt = 0, Nh = 0;
    long long Vs = 0, V = 0, Vh = 0;
    double beta = 0;
    uint64_t seed = 0, sweep = 0, launches = 0;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    int* th = nullptr;         // internal layout, binary angles
    bool own_th = false;
    char* work = nullptr;      // measurement workspace in use
    size_t work_bytes = 0;
    bool own_work = false;     // library-allocated (grown on demand) vs caller-owned
    float* staging = nullptr;  // canonical device copy for set/get links
    double* scratch = nullptr; // [2*NBLK + 4] plaquette partials and sums
    int* d_bad = nullptr;
    int4* hb_queue = nullptr; // heatbath straggler queue (library-owned)
    int* hb_qcount = nullptr;
    int hb_qcap = 0;          // entries per sub-queue
    int hb_qb = 1;            // thread blocks per sub-queue of k_hb_stragglers (grid = one wave)
    uint32_t* d_sweep = nullptr;      // device copy of the sweep counter for graph replays
    bool d_sweep_stale = true;
    bool use_graphs = false, capturing = false;
    bool use_persist = false; // lattices that live in L2: one cooperative launch per compound sweep (ul_persist.cuh)
    int pvec = 1, pbx = 1, pby = 1, pbz = 1, pgrid = 0;   // its tile shape and the largest co-resident grid
    unsigned* d_bar = nullptr; // grid barrier counter
    unsigned bar_base = 0;
    int zflip = 0;            // alternates per sub-step launch (UpdateArgs::zflip)
    bool zflip_on = true;     // UL_NO_ZFLIP=1 turns the alternation off
    cudaStream_t grp_stream[8] = {};   // slab groups side by side (probe)
    cudaEvent_t grp_ev[9] = {};
    int4* grp_queue[8] = {}; int* grp_qcount[8] = {};
    uint32_t* grp_sweep[8] = {};        // per-stream device copies of the sweep counter (graph replays)
    int grp_n = 0;
    bool hb_local_on = true;            // heatbath launches finish their stragglers in the kernel from a shared-memory queue
                                        // (UL_NO_HB_LOCAL=1, and always with peer halo writes: global queue + k_hb_stragglers)
    int group_streams_n = 4;            // groups side by side per round (ul_set_slab_group's second knob; UL_GROUP_STREAMS)
    std::vector<RoundGraph> round_graphs;
    int dev = 0;              // the CUDA device of this context (entry points switch to it)
    // peer-memory halo writes (ul_set_halo_peers): neighbours' link arrays, own-layer range, stream-ordered flags
    int* peer_dn = nullptr; int* peer_up = nullptr;
    int halo_gl = 0;
    uint32_t* halo_flags = nullptr;      // [0]: sub-steps the shard below has completed, [1]: the shard above (written by them)
    uint32_t* peer_flag_dn = nullptr;    // where this shard reports to the shard below (its flags[1]) / above (its flags[0])
    uint32_t* peer_flag_up = nullptr;
    uint32_t halo_seq = 0;               // sub-steps completed since the peers were set
    std::vector<std::pair<cudaIpcMemHandle_t, void*>> ipc_open;   // neighbours' allocations opened through CUDA IPC
    bool or_tma = false, or_tma_attr = false;   // UL_OR_TMA=1: overrelaxation through the bulk-copy staged kernel
    bool use_pdl = true;      // programmatic dependent launch between the update kernels (UL_NO_PDL=1 turns it off)
    cudaStream_t cap_stream = nullptr;
    std::vector<CachedGraph> graphs;
    uint32_t site_offset = 0; // ul_set_site_offset
    int alg = 0;             // ul_set_update_algorithm: 0 heatbath, 1 Metropolis for the stochastic sweeps
    double met_delta = 3.14159265358979323846;
    int vec = 1, bx = 1, by = 1, bz = 1;
    int sub_hb = 1, sub_or = 3, sub_k = 1;
    int batch_cap = 0;       // ul_set_accum_batch: 0 = default depth
    // open measurement
    bool open = false;
    int d = 0, r_max = 0, n_fp = 0, n_slab = 0, d_out = 0, n_outer = 0;
    long long n_acc = 0;
    int n_comb = 0, n_in_seen = 0, n_inner_acc = 0;   // two-level hooks: outer iterations combined, inner configurations per iteration / since the last combine
    int n_pending = 0;       // configurations tabulated but not yet added to the accumulators
    bool multihit = false;   // ul_set_multihit: sums of T at r >= 2 from multihit temporal links
    bool vac_deferred = false; // no field points: the plaquette column sums are taken once, on the final configuration
    int slab_group = -1;     // ul_set_slab_group: slabs per group of the slab-group-major sub-update loop (0 = off, -1 = auto)
    bool skip_colsum = false; // replayed configurations: their plaquette column sums are already in the vacuum sums
    float* staging2 = nullptr; // second configuration copy (two-level replay)
    float* staging_out = nullptr;        // ul_get_links_async: its own canonical copy, a copy stream and two events, so that the
    cudaStream_t copy_stream = nullptr;  // device-to-host copy runs beside whatever the caller enqueues next (ul_set_links of the
    cudaEvent_t ev_repacked = nullptr;   // next configuration: both directions of the link to the host are busy at once)
    cudaEvent_t ev_out_done = nullptr;
    bool out_pending = false;
    float* staging_in = nullptr;         // ul_set_links_async: the upload of the NEXT configuration on a stream of its own while the
    cudaStream_t in_stream = nullptr;    // current one is being worked on; ul_set_links_commit turns it into the link array
    cudaEvent_t ev_in_done = nullptr;
    bool in_pending = false;
    int* bad_host = nullptr;             // the validation flag of ul_set_links_commit in mapped pinned host memory: reading it back must
    int* bad_dev = nullptr;              // not queue a copy behind a ul_get_links_async that is still using the copy engine
    char* plane_buf = nullptr; // full-plane maps through the transverse DFT: Ohat, group partials, Ghat (library-owned)
    size_t plane_bytes = 0;
    bool plane_fresh = true;   // Ghat holds nothing yet
    bool plane_attr_set = false; // shared-memory limits of the plane kernels raised (per context: the attribute is per device)
    double plane_scale = 0.0;
    int plane_r_max = 0;
    bool replay = false;     // ul_multilevel_replay in progress: no TO sums, fields reduced on the fly in pass 2
    bool acc_fresh = true;   // the inner sums A2, B2 hold nothing yet: the next pass writes instead of adding
    Workspace ws;
    // last result
    bool have = false;
    int res_r_max = 0, res_n_fp = 0, res_n_slab = 0;
    const double2* res_A = nullptr;
    double res_inv = 1.0;
    std::vector<double> corr, field, vacuum;
    std::string err;
};

namespace {

DeviceGuard::DeviceGuard(const ul_ctx* c) {
    int cur = -1;
    if (c && cudaGetDevice(&cur) == cudaSuccess && cur != c->dev && cudaSetDevice(c->dev) == cudaSuccess) prev = cur;
}

std::string g_err;   // errors without a handle

int fail(ul_ctx* c, int code, const std::string& msg) {
    if (c) c->err = msg; else g_err = msg;
    return code;
}
#define UL_CUDA(c, call)                                                                       \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess)                                                                 \
            return fail((c), e_ == cudaErrorMemoryAllocation ? UL_ENOMEM : UL_ECUDA,           \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                   \
    } while (0)

ulk::Geom geom(const ul_ctx* c) {
    ulk::Geom g;
    g.Ns = c->Ns; g.Nh = c->Nh; g.Nt = c->Nt; g.Vs = c->Vs; g.V = c->V; g.Vh = c->Vh;
    return g;
}

int largest_divisor_le(int n, int cap) {
    int best = 1;
    for (int v = 1; v <= n && v <= cap; ++v)
        if (n % v == 0) best = v;
    return best;
}

// update kernels are launched with programmatic stream serialization (ul_update.cuh: pdl_wait)
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(const ul_ctx* c, void (*kernel)(KArgs...), dim3 grid, dim3 block, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = 0; cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = c->use_pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}
template <int KIND, int MU>
cudaError_t launch_update_vec(const ul_ctx* c, const ulk::UpdateArgs& a, dim3 grid, dim3 block) {
    switch (c->vec) {
        case 4: return c->capturing ? launch_pdl(c, ulk::k_update<KIND, MU, 4, true>, grid, block, a) : launch_pdl(c, ulk::k_update<KIND, MU, 4, false>, grid, block, a);
        case 2: return c->capturing ? launch_pdl(c, ulk::k_update<KIND, MU, 2, true>, grid, block, a) : launch_pdl(c, ulk::k_update<KIND, MU, 2, false>, grid, block, a);
        default: return c->capturing ? launch_pdl(c, ulk::k_update<KIND, MU, 1, true>, grid, block, a) : launch_pdl(c, ulk::k_update<KIND, MU, 1, false>, grid, block, a);
    }
}
template <int KIND>
cudaError_t launch_update_mu(const ul_ctx* c, int mu, const ulk::UpdateArgs& a, dim3 grid, dim3 block) {
    switch (mu) {
        case 0: return launch_update_vec<KIND, 0>(c, a, grid, block);
        case 1: return launch_update_vec<KIND, 1>(c, a, grid, block);
        case 2: return launch_update_vec<KIND, 2>(c, a, grid, block);
        default: return launch_update_vec<KIND, 3>(c, a, grid, block);
    }
}

// Stream-ordered flags between neighbouring shards (no kernel spins, no host synchronisation): cuStreamWriteValue32 /
// cuStreamWaitValue32 on words in (peer-mapped) device memory, fetched from the driver at run time (libul.so does not link
// against libcuda, so it still loads on a machine without a driver).
typedef int (*StreamMemOp32)(cudaStream_t, unsigned long long, uint32_t, unsigned int);
StreamMemOp32 stream_memop(const char* name) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult st;
    if (cudaGetDriverEntryPoint(name, &fn, cudaEnableDefault, &st) != cudaSuccess || st != cudaDriverEntryPointSuccess) return nullptr;
    return (StreamMemOp32)fn;
}
int halo_wait(ul_ctx* c) {
    static StreamMemOp32 wait32 = stream_memop("cuStreamWaitValue32");
    if (!wait32) return fail(c, UL_ECUDA, "cuStreamWaitValue32 not available");
    for (int i = 0; i < 2; ++i)                                    // CU_STREAM_WAIT_VALUE_GEQ = 0
        if (wait32(c->stream, (unsigned long long)(uintptr_t)(c->halo_flags + i), c->halo_seq, 0u) != 0) return fail(c, UL_ECUDA, "cuStreamWaitValue32");
    return UL_OK;
}
int halo_signal(ul_ctx* c) {
    static StreamMemOp32 write32 = stream_memop("cuStreamWriteValue32");
    if (!write32) return fail(c, UL_ECUDA, "cuStreamWriteValue32 not available");
    c->halo_seq += 1;
    if (write32(c->stream, (unsigned long long)(uintptr_t)c->peer_flag_dn, c->halo_seq, 0u) != 0 ||
        write32(c->stream, (unsigned long long)(uintptr_t)c->peer_flag_up, c->halo_seq, 0u) != 0)
        return fail(c, UL_ECUDA, "cuStreamWriteValue32");
    return UL_OK;
}

// one sub-step (kind, parity, mu), optionally slab-masked: rows a3-a6
// s_begin <= s < s_end: the slabs (of thickness slab_d) this launch covers; the whole lattice when slab_d = 0
int substep(ul_ctx* c, int kind, int parity, int mu, int slab_d, int s_begin = 0, int s_end = -1) {
    static const char* const names[2][3] = {{"ul:hb_substep", "ul:or_substep", "ul:metropolis_substep"},
                                            {"ul:hb_substep_masked", "ul:or_substep_masked", "ul:metropolis_substep_masked"}};
    NvtxRange range(names[slab_d > 0 ? 1 : 0][kind]);
    int n_t = c->Nt, z0 = 0;
    if (slab_d > 0) {
        if (s_end < 0) s_end = c->Nt / slab_d;
        const int per = mu != 0 ? slab_d - 1 : slab_d;    // layers of a slab this direction updates
        n_t = (s_end - s_begin) * per;
        z0 = s_begin * per;
    }
    if (n_t == 0) return UL_OK;                       // thickness 1: every spatial link is frozen
    const bool halo = c->peer_dn != nullptr && slab_d == 0;
    if (halo) { z0 = c->halo_gl; n_t = c->Nt - 2 * c->halo_gl; }   // own layers only: the ghost layers are written by the neighbours
    ulk::UpdateArgs a;
    a.z0 = z0;
    a.peer_dn = halo ? c->peer_dn : nullptr; a.peer_up = halo ? c->peer_up : nullptr;
    a.halo_gl = c->halo_gl; a.halo_nt = c->Nt - 2 * c->halo_gl;
    if (halo && c->peer_flag_dn) {                                // both neighbours have completed the previous sub-step:
        const int rc = halo_wait(c);                              // their halo writes have landed and they no longer read what this
        if (rc) return rc;                                        // sub-step is about to overwrite in their ghost layers
    }
    a.zflip = c->zflip_on ? (c->zflip ^= 1) : 0;
    a.th = c->th; a.Vh = (int)c->Vh; a.Ns = c->Ns; a.Nh = c->Nh; a.Nt = c->Nt;
    a.parity = parity; a.slab_d = slab_d; a.beta = (float)c->beta;
    a.key0 = (uint32_t)(c->seed & 0xffffffffu); a.key1 = (uint32_t)(c->seed >> 32);
    a.sweep_lo = (uint32_t)(c->sweep & 0xffffffffu); a.sweep_hi = (uint32_t)(c->sweep >> 32); a.sweep_dev = c->d_sweep;
    const dim3 block(c->bx, c->by, 2 * c->bz), grid(c->Nh / c->by, c->Ns / c->bz, n_t);   // by = x2 row PAIRS per block
    a.site_offset = c->site_offset;
    a.queue = c->hb_queue; a.qcount = c->hb_qcount; a.qcap = c->hb_qcap;
    {
        const double units = c->met_delta * (4294967296.0 / 6.283185307179586476925286766559);
        a.met_delta_bt = units >= 2147483647.0 ? 2147483647 : (int)(units + 0.5);
    }
    if (kind == 1 && c->or_tma && c->vec == 4 && c->bz == 1 && !c->capturing && !halo) {       // A/B partner of the direct gather (ul_update_tma.cuh)
        const size_t smem = (size_t)18 * 2 * c->by * c->Nh * sizeof(int);
        if (!c->or_tma_attr) {
            cudaFuncSetAttribute(ulk::k_update_or_tma<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            cudaFuncSetAttribute(ulk::k_update_or_tma<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            cudaFuncSetAttribute(ulk::k_update_or_tma<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            cudaFuncSetAttribute(ulk::k_update_or_tma<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            c->or_tma_attr = true;
        }
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr; cfg.numAttrs = c->use_pdl ? 1 : 0;
        const cudaError_t et = mu == 0 ? cudaLaunchKernelEx(&cfg, ulk::k_update_or_tma<0>, a) : mu == 1 ? cudaLaunchKernelEx(&cfg, ulk::k_update_or_tma<1>, a)
                             : mu == 2 ? cudaLaunchKernelEx(&cfg, ulk::k_update_or_tma<2>, a) : cudaLaunchKernelEx(&cfg, ulk::k_update_or_tma<3>, a);
        if (et != cudaSuccess) return fail(c, UL_ECUDA, std::string("k_update_or_tma launch: ") + cudaGetErrorString(et));
        c->launches += 1;
        return UL_OK;
    }
    if (kind == 0 && c->hb_local_on && !halo) {                   // stragglers finished inside the kernel (ul_persist.cuh)
        cudaError_t el = cudaSuccess;
#define UL_HBL(MU_, VEC_)                                                                                                     \
        el = c->capturing ? launch_pdl(c, ulk::k_update_hb_local<MU_, VEC_, true>, grid, block, a)                            \
                          : launch_pdl(c, ulk::k_update_hb_local<MU_, VEC_, false>, grid, block, a)
#define UL_HBL_MU(VEC_)                                                                                                       \
        do { if (mu == 0) { UL_HBL(0, VEC_); } else if (mu == 1) { UL_HBL(1, VEC_); } else if (mu == 2) { UL_HBL(2, VEC_); } else { UL_HBL(3, VEC_); } } while (0)
        if (c->vec == 4) UL_HBL_MU(4); else if (c->vec == 2) UL_HBL_MU(2); else UL_HBL_MU(1);
#undef UL_HBL_MU
#undef UL_HBL
        if (el != cudaSuccess) return fail(c, UL_ECUDA, std::string("k_update_hb_local launch: ") + cudaGetErrorString(el));
        c->launches += 1;
        return UL_OK;
    }
    const cudaError_t e = kind == 0 ? launch_update_mu<0>(c, mu, a, grid, block)
                        : kind == 1 ? launch_update_mu<1>(c, mu, a, grid, block) : launch_update_mu<2>(c, mu, a, grid, block);
    if (e != cudaSuccess) return fail(c, UL_ECUDA, std::string("k_update launch: ") + cudaGetErrorString(e));
    c->launches += 1;
    if (kind == 0) {                                  // finish the links the heatbath kernel queued
        // grid: the sub-queues in use x enough blocks for ~12 % of the launch's links at one entry per thread, at most one wave
        const long long nblk = (long long)grid.x * grid.y * grid.z;
        const int nq = nblk < ulk::HB_NQ ? (int)nblk : ulk::HB_NQ;
        const long long links = nblk * (long long)(block.x * block.y * block.z) * c->vec;
        long long qb = (links / 8 / nq + 255) / 256;
        qb = qb < 1 ? 1 : (qb > c->hb_qb ? c->hb_qb : qb);
        const dim3 sgrid(nq, (unsigned)qb);
        const cudaError_t es = c->capturing ? launch_pdl(c, ulk::k_hb_stragglers<true>, sgrid, dim3(256), a, mu)
                                            : launch_pdl(c, ulk::k_hb_stragglers<false>, sgrid, dim3(256), a, mu);
        if (es != cudaSuccess) return fail(c, UL_ECUDA, std::string("k_hb_stragglers launch: ") + cudaGetErrorString(es));
        c->launches += 1;
    }
    if (halo && c->peer_flag_dn) return halo_signal(c);
    return UL_OK;
}
int one_sweep(ul_ctx* c, int kind, int slab_d, int s_begin = 0, int s_end = -1) {      // O5: parity outer, direction inner
    for (int parity = 0; parity < 2; ++parity)
        for (int mu = 0; mu < 4; ++mu) {
            const int rc = substep(c, kind, parity, mu, slab_d, s_begin, s_end);
            if (rc) return rc;
        }
    if (kind != 1) {                                  // heatbath and Metropolis sweeps consume the counter
        if (c->capturing) { ulk::k_bump_sweep<<<1, 1, 0, c->stream>>>(c->d_sweep); c->launches += 1; }
        else { c->sweep += 1; c->d_sweep_stale = true; }
    }
    return UL_OK;
}
int compound_direct(ul_ctx* c, int n_hb, int n_or, int slab_d, int s_begin = 0, int s_end = -1) {
    for (int i = 0; i < n_hb; ++i) { const int rc = one_sweep(c, c->alg == 1 ? 2 : 0, slab_d, s_begin, s_end); if (rc) return rc; }
    for (int i = 0; i < n_or; ++i) { const int rc = one_sweep(c, 1, slab_d, s_begin, s_end); if (rc) return rc; }
    return UL_OK;
}

// Small lattices (the paper's 24^3 x Nt) are launch-bound: ~5 us per launch against ~1 us of work.  There a
// compound sweep (8 (n_hb + n_or) sub-steps, straggler kernels, counter bump) is captured ONCE per recipe into a
// CUDA graph -- on a side stream, with kernels that read the sweep counter from device memory, so that the graph
// never changes -- and replayed on the caller's stream.  Same kernels, same arithmetic, same results.
// One cooperative launch for the whole compound sweep (ul_persist.cuh)
int compound_persistent(ul_ctx* c, int n_hb, int n_or, int slab_d) {
    NvtxRange range("ul:compound_sweep_persistent");
    ulk::PersistArgs a;
    a.u = ulk::UpdateArgs();
    a.u.th = c->th; a.u.Vh = (int)c->Vh; a.u.Ns = c->Ns; a.u.Nh = c->Nh; a.u.Nt = c->Nt;
    a.u.parity = 0; a.u.slab_d = slab_d; a.u.z0 = 0; a.u.zflip = 0; a.u.beta = (float)c->beta;
    a.u.key0 = (uint32_t)(c->seed & 0xffffffffu); a.u.key1 = (uint32_t)(c->seed >> 32);
    a.u.sweep_lo = (uint32_t)(c->sweep & 0xffffffffu); a.u.sweep_hi = (uint32_t)(c->sweep >> 32); a.u.sweep_dev = nullptr;
    a.u.queue = nullptr; a.u.qcount = nullptr; a.u.qcap = 0;
    a.u.site_offset = c->site_offset;
    {
        const double units = c->met_delta * (4294967296.0 / 6.283185307179586476925286766559);
        a.u.met_delta_bt = units >= 2147483647.0 ? 2147483647 : (int)(units + 0.5);
    }
    a.n_hb = n_hb; a.n_or = n_or; a.stoch_kind = c->alg == 1 ? 2 : 0;
    a.gx = c->Nh / c->pby; a.gy = c->Ns / c->pbz;
    a.nt_time = c->Nt; a.nt_space = slab_d > 0 ? c->Nt / slab_d * (slab_d - 1) : c->Nt;
    const int tiles = a.gx * a.gy * c->Nt;
    const int grid = tiles < c->pgrid ? tiles : c->pgrid;
    a.bar = c->d_bar; a.bar_base = c->bar_base;
    const dim3 block(c->pbx, c->pby, 2 * c->pbz);
    void* args[] = {&a};
    const void* fn = c->pvec == 4 ? (const void*)ulk::k_sweep_persistent<4> : c->pvec == 2 ? (const void*)ulk::k_sweep_persistent<2>
                                                                                             : (const void*)ulk::k_sweep_persistent<1>;
    const cudaError_t e = cudaLaunchCooperativeKernel(fn, dim3(grid), block, args, 0, c->stream);
    if (e != cudaSuccess) return fail(c, UL_ECUDA, std::string("k_sweep_persistent launch: ") + cudaGetErrorString(e));
    c->bar_base += 8u * (unsigned)(n_hb + n_or);
    c->sweep += (uint64_t)n_hb;
    c->d_sweep_stale = true;
    c->launches += 1;
    return UL_OK;
}

int compound(ul_ctx* c, int n_hb, int n_or, int slab_d) {
    if (c->peer_dn != nullptr && slab_d == 0) return compound_direct(c, n_hb, n_or, slab_d);   // halo writes: direct launches
    if (c->use_persist && n_hb + n_or > 0) return compound_persistent(c, n_hb, n_or, slab_d);
    if (!c->use_graphs || n_hb + n_or == 0) return compound_direct(c, n_hb, n_or, slab_d);
    GraphKey key{n_hb, n_or, slab_d, c->alg, c->beta, c->met_delta, c->site_offset};
    CachedGraph* g = nullptr;
    for (auto& e : c->graphs) if (e.key == key) g = &e;
    if (!g) {
        cudaStream_t user = c->stream;
        const uint64_t launches0 = c->launches;
        c->stream = c->cap_stream; c->capturing = true;
        cudaGraph_t graph = nullptr;
        int rc = UL_OK;
        if (cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) rc = UL_ECUDA;
        if (!rc) rc = compound_direct(c, n_hb, n_or, slab_d);
        const cudaError_t ee = cudaStreamEndCapture(c->cap_stream, &graph);
        c->stream = user; c->capturing = false;
        CachedGraph ng;
        ng.key = key; ng.launches = c->launches - launches0;
        c->launches = launches0;
        if (rc || ee != cudaSuccess || !graph || cudaGraphInstantiate(&ng.exec, graph, 0) != cudaSuccess) {
            if (graph) cudaGraphDestroy(graph);
            cudaGetLastError();
            c->use_graphs = false;                    // no graphs on this context: launch directly (same kernels)
            return compound_direct(c, n_hb, n_or, slab_d);
        }
        cudaGraphDestroy(graph);
        if (c->graphs.size() >= 16) {                 // e.g. a scan in beta: keep the cache bounded, drop the oldest recipe
            cudaStreamSynchronize(c->stream);
            cudaGraphExecDestroy(c->graphs.front().exec);
            c->graphs.erase(c->graphs.begin());
        }
        c->graphs.push_back(ng);
        g = &c->graphs.back();
    }
    if (c->d_sweep_stale) {
        ulk::k_set_sweep<<<1, 1, 0, c->stream>>>(c->d_sweep, (uint32_t)(c->sweep & 0xffffffffu), (uint32_t)(c->sweep >> 32));
        c->d_sweep_stale = false;
    }
    if (cudaGraphLaunch(g->exec, c->stream) != cudaSuccess) return fail(c, UL_ECUDA, "cudaGraphLaunch");
    c->sweep += (uint64_t)n_hb;                       // the graph bumped the device counter n_hb times
    c->launches += g->launches;
    return UL_OK;
}

int group_streams(ul_ctx* c, int S) {
    for (; c->grp_n < S; ++c->grp_n) {
        const int k = c->grp_n;
        void* q = nullptr;
        if (cudaStreamCreateWithFlags(&c->grp_stream[k], cudaStreamNonBlocking) != cudaSuccess) return UL_ECUDA;
        if (cudaEventCreateWithFlags(&c->grp_ev[1 + k], cudaEventDisableTiming) != cudaSuccess) return UL_ECUDA;
        if (k == 0 && cudaEventCreateWithFlags(&c->grp_ev[0], cudaEventDisableTiming) != cudaSuccess) return UL_ECUDA;
        if (cudaMalloc(&q, sizeof(int4) * (size_t)ulk::HB_NQ * c->hb_qcap + sizeof(int) * (ulk::HB_NQ + 1)) != cudaSuccess) return UL_ENOMEM;
        c->grp_queue[k] = (int4*)q;
        c->grp_qcount[k] = (int*)(c->grp_queue[k] + (size_t)ulk::HB_NQ * c->hb_qcap);
        if (cudaMemset(c->grp_qcount[k], 0, sizeof(int) * (ulk::HB_NQ + 1)) != cudaSuccess) return UL_ECUDA;
        void* sw = nullptr;
        if (cudaMalloc(&sw, 2 * sizeof(uint32_t)) != cudaSuccess) return UL_ENOMEM;
        c->grp_sweep[k] = (uint32_t*)sw;
    }
    return UL_OK;
}

int accumulate(ul_ctx* c, int s_begin = 0, int s_end = -1);
int flush(ul_ctx* c, int s_begin = 0, int s_end = -1);

// The whole n_sub loop of one ROUND of slab groups (slabs g0 <= s < g1: S groups of grp slabs side by side), captured ONCE as a
// graph and replayed: per sub-update a fork to the group streams (each with its own straggler queue and sweep-counter copy; the
// kernels read the sweep counter from device memory, so the graph never changes), the compound sub-update of every group, a
// join, the round's tables, and an accumulation pass whenever the batch is full.  Leaves the host state as the launches would.
int round_run(ul_ctx* c, int d, int g0, int g1, int grp, int S, int n_sub) {
    RoundGraph* g = nullptr;
    for (auto& e : c->round_graphs)
        if (e.g0 == g0 && e.grp == grp && e.S == S && e.n_hb == c->sub_hb && e.n_or == c->sub_or && e.sub_k == c->sub_k && e.slab_d == d &&
            e.alg == c->alg && e.beta == c->beta && e.met_delta == c->met_delta && e.site_offset == c->site_offset && e.n_sub == n_sub &&
            e.kb == c->ws.kb && e.r_max == c->r_max && e.n_fp == c->n_fp && e.multihit == (c->multihit ? 1 : 0) && e.work == c->work &&
            e.ws_total == c->ws.total) g = &e;
    const bool deferred = c->n_fp == 0 && !c->multihit;             // accumulate(): the vacuum sums are then taken at the end
    if (!g) {
        if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(c, UL_ECUDA, "capture stream");
        cudaStream_t user = c->stream;
        int4* q0 = c->hb_queue; int* qc0 = c->hb_qcount; uint32_t* ds0 = c->d_sweep;
        const uint64_t launches0 = c->launches, sweep_keep = c->sweep;
        cudaGraph_t graph = nullptr;
        int rc = UL_OK;
        if (cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) rc = UL_ECUDA;
        c->capturing = true;
        c->acc_fresh = true; c->n_pending = 0;
        for (int j = 0; j < n_sub && !rc; ++j) {
            if (cudaEventRecord(c->grp_ev[0], c->cap_stream) != cudaSuccess) rc = UL_ECUDA;
            for (int k = 0; k < S && !rc; ++k) {
                const int s0 = g0 + k * grp;
                if (s0 >= g1) break;
                const int s1 = s0 + grp < g1 ? s0 + grp : g1;
                if (cudaStreamWaitEvent(c->grp_stream[k], c->grp_ev[0], 0) != cudaSuccess) { rc = UL_ECUDA; break; }
                c->stream = c->grp_stream[k]; c->hb_queue = c->grp_queue[k]; c->hb_qcount = c->grp_qcount[k]; c->d_sweep = c->grp_sweep[k];
                for (int kk = 0; kk < c->sub_k && !rc; ++kk) rc = compound_direct(c, c->sub_hb, c->sub_or, d, s0, s1);
                if (!rc && deferred) rc = accumulate(c, s0, s1);    // U table only: the group's own table launch, on its stream
                if (!rc && (cudaEventRecord(c->grp_ev[1 + k], c->grp_stream[k]) != cudaSuccess ||
                            cudaStreamWaitEvent(c->cap_stream, c->grp_ev[1 + k], 0) != cudaSuccess)) rc = UL_ECUDA;
            }
            c->stream = c->cap_stream; c->hb_queue = q0; c->hb_qcount = qc0; c->d_sweep = ds0;
            if (!rc && !deferred) rc = accumulate(c, g0, g1);       // tables with plaquettes (shared partial sums): after the join
            if (!rc) {
                c->n_pending += 1;
                if (c->n_pending == c->ws.kb || j == n_sub - 1) rc = flush(c, g0, g1);
            }
        }
        const cudaError_t ee = cudaStreamEndCapture(c->cap_stream, &graph);
        c->stream = user; c->hb_queue = q0; c->hb_qcount = qc0; c->d_sweep = ds0; c->capturing = false;
        c->sweep = sweep_keep;
        RoundGraph ng;
        ng.g0 = g0; ng.grp = grp; ng.S = S; ng.n_hb = c->sub_hb; ng.n_or = c->sub_or; ng.sub_k = c->sub_k; ng.slab_d = d; ng.alg = c->alg;
        ng.n_sub = n_sub; ng.kb = c->ws.kb; ng.r_max = c->r_max; ng.n_fp = c->n_fp; ng.multihit = c->multihit ? 1 : 0;
        ng.work = c->work; ng.ws_total = c->ws.total;
        ng.beta = c->beta; ng.met_delta = c->met_delta; ng.site_offset = c->site_offset;
        ng.launches = c->launches - launches0;
        c->launches = launches0;
        if (rc || ee != cudaSuccess || !graph || cudaGraphInstantiate(&ng.exec, graph, 0) != cudaSuccess) {
            if (graph) cudaGraphDestroy(graph);
            cudaGetLastError();
            return fail(c, UL_ECUDA, "slab-group round: graph capture failed");
        }
        cudaGraphDestroy(graph);
        if (c->round_graphs.size() >= 32) {                            // bounded cache
            cudaStreamSynchronize(c->stream);
            cudaGraphExecDestroy(c->round_graphs.front().exec);
            c->round_graphs.erase(c->round_graphs.begin());
        }
        c->round_graphs.push_back(ng);
        g = &c->round_graphs.back();
    }
    if (cudaGraphLaunch(g->exec, c->stream) != cudaSuccess) return fail(c, UL_ECUDA, "cudaGraphLaunch (slab-group round)");
    c->sweep += (uint64_t)c->sub_hb * (uint64_t)c->sub_k * (uint64_t)n_sub;
    c->launches += g->launches;
    c->n_pending = 0; c->acc_fresh = false;
    if (deferred) c->vac_deferred = true;
    return UL_OK;
}

// slabs per group of the slab-group-major sub-update loop; 0 = sub-update-major (one launch over all slabs)
int slab_group_size(const ul_ctx* c, int d) {
    if (c->slab_group >= 0) return c->slab_group;
    // auto: lattices whose links do not fit L2 -- rounds of ~64 MB of links (4 links x 4 B per site) in flight, split over the
    // group streams; measured on 64^4, d = 2: 8 slabs in flight (4 x 2 or 2 x 4) are the optimum, 12.6 % faster than one launch
    // over all slabs, 6 or 12 slabs are 2-4 % behind it
    const double link_bytes = 16.0 * (double)c->V;
    if (link_bytes <= 96e6) return 0;
    const double per_slab = 16.0 * (double)c->Vs * d;
    const int S = c->group_streams_n > 1 ? c->group_streams_n : 1;
    int g = (int)(64e6 / per_slab / S + 0.5);
    if (g < 1) g = 1;
    while (g > 1 && c->n_slab % (g * S) != 0) --g;                     // whole rounds where possible
    if (2 * g * S > c->n_slab) return 0;                               // not even two rounds: nothing to keep resident
    return g;
}

int check_meas_args(ul_ctx* c, int d, int r_max, const int* fps, int n_fp) {
    if (d < 1 || c->Nt % d != 0) return fail(c, UL_EINVAL, "Nt % slab_thickness != 0");
    if (r_max < 1 || r_max > c->Ns / 2) return fail(c, UL_EINVAL, "r_max out of range [1, Ns/2]");
    if (n_fp < 0 || (n_fp > 0 && !fps)) return fail(c, UL_EINVAL, "bad field points");
    return UL_OK;
}

template <typename T> T* wsp(ul_ctx* c, size_t off) { return reinterpret_cast<T*>(c->work + off); }

// reserve the workspace, upload the field points, zero the accumulators
int open_measurement(ul_ctx* c, int d_in, int d_out, int r_max, const int* fps, int n_fp) {
    const Workspace w = plan_workspace(c->Ns, c->Nt, d_in, d_out, r_max, n_fp, c->replay, c->multihit);
    if (w.total > c->work_bytes) {
        if (!c->own_work && c->work) return fail(c, UL_ENOMEM, "accumulators exceed the caller's workspace");
        if (c->work) { UL_CUDA(c, cudaStreamSynchronize(c->stream)); cudaFree(c->work); c->work = nullptr; c->work_bytes = 0; }
        void* p = nullptr;
        UL_CUDA(c, cudaMalloc(&p, w.total));
        c->work = (char*)p; c->work_bytes = w.total; c->own_work = true;
    }
    c->ws = w;
    if (c->batch_cap > 0 && c->batch_cap < c->ws.kb) c->ws.kb = c->batch_cap;
    c->d = d_in; c->d_out = d_out; c->r_max = r_max; c->n_fp = n_fp;
    c->n_slab = c->Nt / d_in; c->n_outer = d_out > 0 ? c->Nt / d_out : 0;
    c->n_acc = 0;
    c->n_pending = 0;
    c->acc_fresh = true;
    c->plane_fresh = true;
    c->vac_deferred = false;
    c->have = false;
    if (n_fp > 0) UL_CUDA(c, cudaMemcpyAsync(c->work + w.fps, fps, sizeof(int) * 3 * (size_t)n_fp, cudaMemcpyHostToDevice, c->stream));
    if (w.partial > w.A4) UL_CUDA(c, cudaMemsetAsync(c->work + w.A4, 0, w.partial - w.A4, c->stream));   // A4, B4 (A2, B2: first pass writes)
    UL_CUDA(c, cudaMemsetAsync(c->work + w.result, 0, w.total - w.result, c->stream));
    if (n_fp > 0) UL_CUDA(c, cudaStreamSynchronize(c->stream));                            // fps is a caller-owned host buffer
    c->open = true;
    return UL_OK;
}

double* res_colsum(ul_ctx* c) { return wsp<double>(c, c->ws.result) + 2 * (size_t)c->r_max * (1 + 12 * (size_t)c->n_fp) + 12; }
double* res_vacuum(ul_ctx* c) { return wsp<double>(c, c->ws.result) + 2 * (size_t)c->r_max * (1 + 12 * (size_t)c->n_fp); }

// adds the tabulated configurations (slots 0..n_pending-1) to the accumulators: rows a7, a8
// (restricted to the slabs s_begin <= s < s_end when s_end >= 0: slab-group-major order)
int flush(ul_ctx* c, int s_begin, int s_end) {
    if (c->n_pending == 0) return UL_OK;
    NvtxRange range("ul:accumulate_batch");
    if (s_end < 0) s_end = c->n_slab;
    const long long n = (long long)(s_end - s_begin) * c->Vs;
    const int nb = (int)((n + 255) / 256);
    ulk::AccumArgs a;
    a.idx0 = (long long)s_begin * c->Vs; a.n_idx = n;
    a.g = geom(c); a.d = c->d; a.n_slab = c->n_slab; a.r_max = c->r_max; a.n_fp = c->n_fp; a.nk = c->n_pending; a.first = c->acc_fresh ? 1 : 0;
    a.U = wsp<double2>(c, c->ws.U); a.Ot = wsp<float>(c, c->ws.Ot); a.fps = wsp<int>(c, c->ws.fps);
    a.A = wsp<double2>(c, c->ws.A2); a.B = wsp<double2>(c, c->ws.B2);
#define UL_ACC_LAUNCH(KB, FIELD)                                                                     \
    do {                                                                                            \
        if (a.nk == KB) ulk::k_accumulate<KB, FIELD, true><<<nb, 256, 0, c->stream>>>(a);           \
        else ulk::k_accumulate<KB, FIELD, false><<<nb, 256, 0, c->stream>>>(a);                     \
        c->launches += 1;                                                                           \
    } while (0)
    const bool fields = c->n_fp > 0 && !c->replay;
    auto launch = [&](bool with_fields) {
        if (with_fields) {
            if (a.nk == 1) UL_ACC_LAUNCH(1, true);
            else if (a.nk <= 4) UL_ACC_LAUNCH(4, true);
            else UL_ACC_LAUNCH(KBATCH, true);
        } else {
            if (a.nk == 1) UL_ACC_LAUNCH(1, false);
            else if (a.nk <= 4) UL_ACC_LAUNCH(4, false);
            else UL_ACC_LAUNCH(KBATCH, false);
        }
    };
    a.r_begin = 1; a.r_end = c->r_max; a.a_r_max = c->r_max;
    if (!c->multihit) {
        launch(fields);
    } else {
        // multihit: the sums of T at r >= 2 come from the Um tables; r = 1 (the two lines share plaquettes) and every
        // TO sum keep the plain T
        if (fields) { a.a_r_max = 1; launch(true); }                                    // TO for all r, T for r = 1
        else { a.r_end = 1; launch(false); }                                             // T for r = 1
        if (c->r_max >= 2) {
            a.U = wsp<double2>(c, c->ws.Um);
            a.r_begin = 2; a.r_end = c->r_max; a.a_r_max = c->r_max;
            launch(false);                                                               // T for r >= 2
        }
    }
#undef UL_ACC_LAUNCH
    UL_CUDA(c, cudaGetLastError());
    c->n_pending = 0;
    c->acc_fresh = false;
    return UL_OK;
}

// the plaquette column sums of the current configuration, added to the vacuum sums (no table is written)
int vacuum_pass(ul_ctx* c) {
    ulk::TableArgs t;
    t.g = geom(c); t.th = c->th; t.d = c->d; t.n_slab = c->n_slab;
    t.U = nullptr; t.Um = nullptr; t.beta = (float)c->beta; t.Ot = nullptr;
    t.partial = wsp<double>(c, c->ws.partial);
    t.row0 = 0; t.n_rows = c->n_slab * c->Ns;
    const int gx = (c->Ns * c->Ns + 255) / 256, rows = t.n_rows;
    const int gy = rows < TBLK / gx ? rows : (TBLK / gx > 0 ? TBLK / gx : 1);
    ulk::k_slab_tables<<<dim3(gx, gy), 256, 0, c->stream>>>(t);
    ulk::k_sum_partials<<<12, 256, 0, c->stream>>>(t.partial, gx * gy, res_colsum(c), 1.0, 1);
    UL_CUDA(c, cudaGetLastError());
    c->launches += 2;
    return UL_OK;
}

// tabulates the current configuration (U, Ot, column sums of O) into the next batch slot; the batch is
// added to the accumulators when it is full, and before anything reads them.  With a slab range (s_end >= 0) only
// those slabs are tabulated, and the caller counts the configuration and flushes (slab-group-major order).
int accumulate(ul_ctx* c, int s_begin, int s_end) {
    NvtxRange range("ul:slab_tables");
    const bool ranged = s_end >= 0;
    if (!ranged) s_end = c->n_slab;
    const long long n = (long long)c->n_slab * c->Vs;
    ulk::TableArgs t;
    t.g = geom(c); t.th = c->th; t.d = c->d; t.n_slab = c->n_slab;
    t.U = wsp<double2>(c, c->ws.U) + (size_t)c->n_pending * n;
    t.Um = c->multihit ? wsp<double2>(c, c->ws.Um) + (size_t)c->n_pending * n : nullptr;
    t.beta = (float)c->beta;
    t.Ot = (c->n_fp > 0 && !c->replay) ? wsp<float>(c, c->ws.Ot) + (size_t)c->n_pending * 12 * n : nullptr;
    t.partial = wsp<double>(c, c->ws.partial);
    t.row0 = s_begin * c->Ns; t.n_rows = (s_end - s_begin) * c->Ns;
    if (c->n_fp == 0 && !c->multihit) {
        // nothing needs the plaquettes: U table only (row a7); the vacuum values are then taken on the final
        // configuration of the measurement (finish())
        const long long threads = (long long)t.n_rows * c->Ns * c->Nh;
        ulk::k_slab_tables_u<<<(unsigned)((threads + 255) / 256), 256, 0, c->stream>>>(t);
        c->vac_deferred = true;
    } else {
        const int gx = (c->Ns * c->Ns + 255) / 256, rows = t.n_rows;
        const int gy = rows < TBLK / gx ? rows : (TBLK / gx > 0 ? TBLK / gx : 1);
        ulk::k_slab_tables<<<dim3(gx, gy), 256, 0, c->stream>>>(t);
        if (!c->skip_colsum) { ulk::k_sum_partials<<<12, 256, 0, c->stream>>>(t.partial, gx * gy, res_colsum(c), 1.0, 1); c->launches += 1; }
    }
    UL_CUDA(c, cudaGetLastError());
    c->launches += 1;
    if (ranged) return UL_OK;
    c->n_acc += 1;
    c->n_pending += 1;
    if (c->n_pending == c->ws.kb) return flush(c);
    return UL_OK;
}

// row a10 on accumulators (A, B) with n_slab slabs, scaled by inv; results to the host vectors
int finish(ul_ctx* c, const double2* A, const double2* B, int n_slab, double inv, double vac_inv) {
    NvtxRange range("ul:slab_product");
    const int R = c->r_max, F = c->n_fp;
    const int n_entries = R * (1 + 12 * F);
    ulk::ReduceArgs a;
    a.Vs = c->Vs; a.r_max = R; a.n_fp = F; a.n_slab = n_slab; a.inv = inv; a.A = A; a.B = B;
    a.partial = wsp<double>(c, c->ws.partial);
    ulk::k_slab_product<false><<<dim3(NBLK, R), 256, 0, c->stream>>>(a, 0);
    const bool stored = F > 0 && !c->replay;       // replay: the field sums were reduced on the fly into the result buffer
    if (stored) { ulk::k_slab_product<true><<<dim3(NBLK, n_entries - R), 256, 0, c->stream>>>(a, R); c->launches += 1; }
    double* res = wsp<double>(c, c->ws.result);
    // C /= 3 Vs ; G /= 3 Vs Nt (DESIGN R9)
    ulk::k_sum_partials<<<2 * R, 256, 0, c->stream>>>(a.partial, NBLK, res, 1.0 / (3.0 * (double)c->Vs), 0);
    c->launches += 2;
    if (stored) {
        ulk::k_sum_partials<<<2 * (n_entries - R), 256, 0, c->stream>>>(a.partial + (size_t)2 * R * NBLK, NBLK, res + 2 * R,
                                                                        1.0 / (3.0 * (double)c->Vs * (double)c->Nt), 0);
        c->launches += 1;
    }
    if (c->vac_deferred) {                          // no field points: vacuum values of the final configuration (include/ul.h)
        const int rc = vacuum_pass(c);
        if (rc) return rc;
        vac_inv = 1.0;
        c->vac_deferred = false;
    }
    ulk::k_vacuum<<<1, 32, 0, c->stream>>>(res_colsum(c), vac_inv / (3.0 * (double)c->V), res_vacuum(c));
    c->launches += 1;
    UL_CUDA(c, cudaGetLastError());
    std::vector<double> host((size_t)2 * n_entries + 12);
    UL_CUDA(c, cudaMemcpyAsync(host.data(), res, sizeof(double) * host.size(), cudaMemcpyDeviceToHost, c->stream));
    UL_CUDA(c, cudaStreamSynchronize(c->stream));
    c->corr.assign(host.begin(), host.begin() + 2 * R);
    c->field.assign(host.begin() + 2 * R, host.begin() + 2 * n_entries);
    c->vacuum.assign(host.begin() + 2 * n_entries, host.end());
    c->res_r_max = R; c->res_n_fp = F; c->res_n_slab = n_slab; c->res_A = A; c->res_inv = inv;
    c->have = true;
    c->open = false;
    return UL_OK;
}

int create_common(ul_ctx** h, int Ns, int Nt, double beta, uint64_t seed, void* dev_links, size_t links_bytes,
                  void* dev_work, size_t work_bytes, void* stream, bool ext) {
    if (!h) return fail(nullptr, UL_EINVAL, "null handle pointer");
    *h = nullptr;
    if (Ns < 2 || Nt < 2 || (Ns & 1) || (Nt & 1) || !(beta >= 0.0)) return fail(nullptr, UL_EINVAL, "need even Ns, Nt >= 2 and beta >= 0");
    const int Nh = Ns / 2;
    const int vec = (Nh % 4 == 0) ? 4 : ((Nh % 2 == 0) ? 2 : 1);
    if (Nh / vec > 128 || 4.0 * (double)Ns * Ns * Ns * Nt >= 2147483648.0) return fail(nullptr, UL_EINVAL, "lattice too large for this build");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return fail(nullptr, UL_ECUDA, "no CUDA device");
    ul_ctx* c = new (std::nothrow) ul_ctx;
    if (!c) return fail(nullptr, UL_ENOMEM, "host allocation failed");
    cudaGetDevice(&c->dev);
    c->Ns = Ns; c->Nt = Nt; c->Nh = Nh;
    c->Vs = (long long)Ns * Ns * Ns; c->V = c->Vs * Nt; c->Vh = c->V / 2;
    c->beta = beta; c->seed = seed;
    c->vec = vec; c->bx = Nh / vec;
    // A block's 128 row pairs are split evenly between x2 and x3 (64^4: 4 x2 row pairs x 4 x3 layers; neighbours displaced in x2
    // AND in x3 are then found in L1): OR sweep 406 -> 396 us, masked compound sub-update 1.64 -> 1.63 ms on 64^4 against all
    // 16 row pairs along x2 (8 x 2: 400 us; 2 x 8: 406 us)
    { int r = 1; while ((r + 1) * (r + 1) <= 128 / c->bx) ++r; c->by = largest_divisor_le(Nh, r); }   // x2 row pairs per block
    c->bz = largest_divisor_le(Ns, 128 / (c->bx * c->by));
    { const char* e = getenv("UL_BLOCK_BY");                         // A/B switch: x2 row pairs per block (the rest of the 128 goes to x3)
      if (e) { const int v = atoi(e); if (v >= 1 && Nh % v == 0 && v * c->bx <= 128) { c->by = v; c->bz = largest_divisor_le(Ns, 128 / (c->bx * c->by)); } } }
    const size_t need = sizeof(float) * 4 * (size_t)c->V;
    if (ext) {
        if (!dev_links || links_bytes < need || ((uintptr_t)dev_links & 255)) { delete c; return fail(nullptr, UL_EINVAL, "dev_links too small or misaligned"); }
        c->th = (int*)dev_links;
        c->stream = (cudaStream_t)stream;
        if (dev_work && work_bytes) { c->work = (char*)dev_work; c->work_bytes = work_bytes; c->own_work = false; }
        else c->own_work = true;
    } else {
        void* p = nullptr;
        cudaError_t e = cudaMalloc(&p, need);
        if (e != cudaSuccess) { delete c; return fail(nullptr, UL_ENOMEM, std::string("cudaMalloc links: ") + cudaGetErrorString(e)); }
        c->th = (int*)p; c->own_th = true;
        e = cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) { cudaFree(p); delete c; return fail(nullptr, UL_ECUDA, std::string("cudaStreamCreate: ") + cudaGetErrorString(e)); }
        c->own_stream = true; c->own_work = true;
    }
    void* s = nullptr;
    if (cudaMalloc(&s, sizeof(double) * (2 * NBLK + 4) + 256) != cudaSuccess) { ul_destroy(c); return fail(nullptr, UL_ENOMEM, "cudaMalloc scratch"); }
    c->scratch = (double*)s;
    c->d_bad = (int*)((char*)s + sizeof(double) * (2 * NBLK + 4));
    // heatbath straggler queue: HB_NQ compact sub-queues, together a quarter of the links of a sub-step (8-12 % are used)
    c->hb_qcap = (int)(c->Vh / 4 / ulk::HB_NQ);
    if (c->hb_qcap < 256) c->hb_qcap = 256;
    {
        int dev = 0, sms = 148, per_sm = 4;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ulk::k_hb_stragglers<false>, 256, 0) != cudaSuccess || per_sm < 1) per_sm = 4;
        c->hb_qb = sms * per_sm / ulk::HB_NQ;
        if (c->hb_qb < 1) c->hb_qb = 1;
    }
    void* q = nullptr;
    if (cudaMalloc(&q, sizeof(int4) * (size_t)ulk::HB_NQ * c->hb_qcap + sizeof(int) * (ulk::HB_NQ + 1)) != cudaSuccess) { ul_destroy(c); return fail(nullptr, UL_ENOMEM, "cudaMalloc straggler queue"); }
    c->hb_queue = (int4*)q;
    c->hb_qcount = (int*)(c->hb_queue + (size_t)ulk::HB_NQ * c->hb_qcap);
    if (cudaMemset(c->hb_qcount, 0, sizeof(int) * (ulk::HB_NQ + 1)) != cudaSuccess) { ul_destroy(c); return fail(nullptr, UL_ECUDA, "memset straggler counters"); }
    c->d_sweep = (uint32_t*)(c->d_bad + 2);
    { const char* e = getenv("UL_NO_ZFLIP"); if (e && e[0] == '1') c->zflip_on = false; }
    { const char* e = getenv("UL_NO_HB_LOCAL"); if (e && e[0] == '1') c->hb_local_on = false; }
    { const char* e = getenv("UL_GROUP_STREAMS"); if (e) { const int v = atoi(e); c->group_streams_n = v < 1 ? 1 : (v > 8 ? 8 : v); } }
    { const char* e = getenv("UL_OR_TMA");                           // the staged kernel works on blocks of one x3 layer: all row pairs along x2
      if (e && e[0] == '1') {
          const int by = largest_divisor_le(Nh, 128 / c->bx), bz = largest_divisor_le(Ns, 128 / (c->bx * by));
          if (bz == 1 && 18 * 2 * by * c->Nh * 4 <= 200 * 1024) { c->by = by; c->bz = bz; c->or_tma = true; }
      } }
    { const char* e = getenv("UL_NO_PDL"); if (e && e[0] == '1') c->use_pdl = false; }
    c->use_graphs = c->V <= (1LL << 21) && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) == cudaSuccess;
    // persistent compound sweeps: tiles with shorter per-thread chains (2 links per thread) than the streaming kernels
    if (c->V <= (1LL << 21)) {
        const char* env = getenv("UL_PERSIST_VEC");
        int pv = env ? atoi(env) : 2;
        if (pv != 1 && pv != 2 && pv != 4) pv = 2;
        while (pv > 1 && c->Nh % pv != 0) pv >>= 1;
        c->pvec = pv; c->pbx = Nh / pv;
        if (c->pbx <= 128) {
            c->pby = largest_divisor_le(Nh, 128 / c->pbx);
            c->pbz = largest_divisor_le(Ns, 128 / (c->pbx * c->pby));
            int dev = 0, sms = 0, per_sm = 0, coop = 0;
            cudaGetDevice(&dev);
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
            const void* fn = pv == 4 ? (const void*)ulk::k_sweep_persistent<4> : pv == 2 ? (const void*)ulk::k_sweep_persistent<2>
                                                                                         : (const void*)ulk::k_sweep_persistent<1>;
            const int threads = c->pbx * c->pby * 2 * c->pbz;
            const long long tiles = (long long)(Nh / c->pby) * (Ns / c->pbz) * Nt;
            if (coop && tiles <= ulk::PERSIST_MAX_TILES && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, threads, 0) == cudaSuccess && per_sm > 0) {
                c->pgrid = sms * per_sm;
                const size_t bar_bytes = 128;
                void* bp = nullptr;
                const char* off = getenv("UL_NO_PERSIST");
                if (!(off && off[0] == '1') && cudaMalloc(&bp, bar_bytes) == cudaSuccess) {
                    c->d_bar = (unsigned*)bp;
                    c->use_persist = cudaMemset(c->d_bar, 0, bar_bytes) == cudaSuccess;
                }
            }
            cudaGetLastError();
        }
    }
    *h = c;
    const int rc = ul_init(c, 1);
    if (rc) { g_err = c->err; ul_destroy(c); *h = nullptr; }
    return rc;
}

}  // namespace

extern "C" {

int ul_create(ul_ctx** h, int Ns, int Nt, double beta, uint64_t seed) {
    return create_common(h, Ns, Nt, beta, seed, nullptr, 0, nullptr, 0, nullptr, false);
}
int ul_create_ext(ul_ctx** h, int Ns, int Nt, double beta, uint64_t seed, void* dev_links, size_t links_bytes,
                  void* dev_work, size_t work_bytes, void* cuda_stream) {
    return create_common(h, Ns, Nt, beta, seed, dev_links, links_bytes, dev_work, work_bytes, cuda_stream, true);
}
size_t ul_workspace_bytes(int Ns, int Nt, int d_in, int d_out, int r_max, int n_fp) {
    if (Ns < 2 || Nt < 2 || d_in < 1 || Nt % d_in != 0 || d_out < 0 || (d_out > 0 && (d_out % d_in != 0 || Nt % d_out != 0)) ||
        r_max < 1 || n_fp < 0)
        return 0;
    return plan_workspace(Ns, Nt, d_in, d_out, r_max, n_fp).total;
}
size_t ul_workspace_bytes_replay(int Ns, int Nt, int d, int r_max, int n_fp) {
    if (Ns < 2 || Nt < 2 || d < 1 || Nt % d != 0 || r_max < 1 || n_fp < 0) return 0;
    return plan_workspace(Ns, Nt, d, 0, r_max, n_fp, n_fp > 0).total;
}
size_t ul_workspace_bytes_replay2(int Ns, int Nt, int d_in, int d_out, int r_max, int n_fp) {
    if (Ns < 2 || Nt < 2 || d_in < 1 || Nt % d_in != 0 || d_out < d_in || d_out % d_in != 0 || Nt % d_out != 0 || r_max < 1 || n_fp < 0) return 0;
    return plan_workspace(Ns, Nt, d_in, d_out, r_max, n_fp, n_fp > 0).total;
}
int ul_destroy(ul_ctx* c) {
    if (!c) return UL_OK;
    DeviceGuard guard(c);
    cudaStreamSynchronize(c->stream);
    if (c->own_th && c->th) cudaFree(c->th);
    if (c->own_work && c->work) cudaFree(c->work);
    if (c->staging) cudaFree(c->staging);
    if (c->staging2) cudaFree(c->staging2);
    if (c->copy_stream) { cudaStreamSynchronize(c->copy_stream); cudaStreamDestroy(c->copy_stream); }
    if (c->ev_repacked) cudaEventDestroy(c->ev_repacked);
    if (c->ev_out_done) cudaEventDestroy(c->ev_out_done);
    if (c->staging_out) cudaFree(c->staging_out);
    if (c->in_stream) { cudaStreamSynchronize(c->in_stream); cudaStreamDestroy(c->in_stream); }
    if (c->ev_in_done) cudaEventDestroy(c->ev_in_done);
    if (c->staging_in) cudaFree(c->staging_in);
    if (c->bad_host) cudaFreeHost(c->bad_host);
    if (c->plane_buf) cudaFree(c->plane_buf);
    if (c->scratch) cudaFree(c->scratch);
    if (c->hb_queue) cudaFree(c->hb_queue);
    if (c->d_bar) cudaFree(c->d_bar);
    for (auto& e : c->ipc_open) cudaIpcCloseMemHandle(e.second);
    for (auto& e : c->round_graphs) if (e.exec) cudaGraphExecDestroy(e.exec);
    for (int k = 0; k < c->grp_n; ++k) {
        if (c->grp_stream[k]) cudaStreamDestroy(c->grp_stream[k]);
        if (c->grp_ev[1 + k]) cudaEventDestroy(c->grp_ev[1 + k]);
        if (c->grp_queue[k]) cudaFree(c->grp_queue[k]);
        if (c->grp_sweep[k]) cudaFree(c->grp_sweep[k]);
    }
    if (c->grp_ev[0]) cudaEventDestroy(c->grp_ev[0]);
    if (c->halo_flags) cudaFree(c->halo_flags);
    for (auto& e : c->graphs) if (e.exec) cudaGraphExecDestroy(e.exec);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    if (c->own_stream && c->stream) cudaStreamDestroy(c->stream);
    delete c;
    return UL_OK;
}

int ul_init(ul_ctx* c, int mode) {
    if (!c || (mode != 0 && mode != 1)) return fail(c, UL_EINVAL, "mode must be 0 or 1");
    DeviceGuard guard(c);
    if (mode == 0) {
        UL_CUDA(c, cudaMemsetAsync(c->th, 0, sizeof(float) * 4 * (size_t)c->V, c->stream));
        return UL_OK;
    }
    const long long n = 4 * c->V;
    ulk::k_hot_start<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(geom(c), c->th, (uint32_t)(c->seed & 0xffffffffu),
                                                                         (uint32_t)(c->seed >> 32));
    UL_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return UL_OK;
}
int ul_set_beta(ul_ctx* c, double beta) {
    if (!c || !(beta >= 0.0)) return fail(c, UL_EINVAL, "beta must be >= 0");
    c->beta = beta;
    return UL_OK;
}

static int ensure_staging(ul_ctx* c) {
    if (c->staging) return UL_OK;
    void* p = nullptr;
    UL_CUDA(c, cudaMalloc(&p, sizeof(float) * 4 * (size_t)c->V));
    c->staging = (float*)p;
    return UL_OK;
}
static int links_in(ul_ctx* c, const void* host, int mode) {
    if (!c || !host) return fail(c, UL_EINVAL, "null pointer");
    DeviceGuard guard(c);
    int rc = ensure_staging(c);
    if (rc) return rc;
    const long long n = 4 * c->V;
    UL_CUDA(c, cudaMemsetAsync(c->d_bad, 0, sizeof(int), c->stream));
    UL_CUDA(c, cudaMemcpyAsync(c->staging, host, sizeof(float) * (size_t)n, cudaMemcpyHostToDevice, c->stream));
    ulk::k_repack<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(geom(c), c->th, c->staging, mode, c->d_bad);
    UL_CUDA(c, cudaGetLastError());
    c->launches += 1;
    int bad = 0;
    UL_CUDA(c, cudaMemcpyAsync(&bad, c->d_bad, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    UL_CUDA(c, cudaStreamSynchronize(c->stream));
    if (bad) return fail(c, UL_EINVAL, "link angles must be finite with |theta| <= 3.2 (wrap them to [-pi, pi] first)");
    return UL_OK;
}
static int links_out(ul_ctx* c, void* host, int mode) {
    if (!c || !host) return fail(c, UL_EINVAL, "null pointer");
    DeviceGuard guard(c);
    int rc = ensure_staging(c);
    if (rc) return rc;
    const long long n = 4 * c->V;
    ulk::k_repack<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(geom(c), c->th, c->staging, mode, c->d_bad);
    UL_CUDA(c, cudaGetLastError());
    c->launches += 1;
    UL_CUDA(c, cudaMemcpyAsync(host, c->staging, sizeof(float) * (size_t)n, cudaMemcpyDeviceToHost, c->stream));
    UL_CUDA(c, cudaStreamSynchronize(c->stream));
    return UL_OK;
}
// The read-back without waiting for it: repack on the context's stream into a buffer of its own, the copy to the host on a
// second stream behind an event.  A following call waits (on the stream) for the previous copy before it overwrites the buffer.
int ul_get_links_async(ul_ctx* c, float* host) {
    if (!c || !host) return fail(c, UL_EINVAL, "null pointer");
    DeviceGuard guard(c);
    const long long n = 4 * c->V;
    if (!c->staging_out) {
        void* p = nullptr;
        UL_CUDA(c, cudaMalloc(&p, sizeof(float) * (size_t)n));
        c->staging_out = (float*)p;
        UL_CUDA(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        UL_CUDA(c, cudaEventCreateWithFlags(&c->ev_repacked, cudaEventDisableTiming));
        UL_CUDA(c, cudaEventCreateWithFlags(&c->ev_out_done, cudaEventDisableTiming));
    }
    if (c->out_pending) UL_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_out_done, 0));
    ulk::k_repack<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(geom(c), c->th, c->staging_out, 0, c->d_bad);
    UL_CUDA(c, cudaGetLastError());
    c->launches += 1;
    UL_CUDA(c, cudaEventRecord(c->ev_repacked, c->stream));
    UL_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->ev_repacked, 0));
    UL_CUDA(c, cudaMemcpyAsync(host, c->staging_out, sizeof(float) * (size_t)n, cudaMemcpyDeviceToHost, c->copy_stream));
    UL_CUDA(c, cudaEventRecord(c->ev_out_done, c->copy_stream));
    c->out_pending = true;
    return UL_OK;
}
int ul_get_links_wait(ul_ctx* c) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    if (!c->out_pending) return UL_OK;
    DeviceGuard guard(c);
    UL_CUDA(c, cudaEventSynchronize(c->ev_out_done));
    c->out_pending = false;
    return UL_OK;
}
// The upload ahead of time: host -> a buffer of its own on a second stream (nothing the context's stream does is touched), and
// the commit that makes it the configuration (repack + validation on the context's stream, behind the upload's event).
int ul_set_links_async(ul_ctx* c, const float* host) {
    if (!c || !host) return fail(c, UL_EINVAL, "null pointer");
    DeviceGuard guard(c);
    const long long n = 4 * c->V;
    if (!c->staging_in) {
        void* p = nullptr;
        UL_CUDA(c, cudaMalloc(&p, sizeof(float) * (size_t)n));
        c->staging_in = (float*)p;
        UL_CUDA(c, cudaStreamCreateWithFlags(&c->in_stream, cudaStreamNonBlocking));
        UL_CUDA(c, cudaEventCreateWithFlags(&c->ev_in_done, cudaEventDisableTiming));
        UL_CUDA(c, cudaHostAlloc((void**)&c->bad_host, sizeof(int), cudaHostAllocMapped));
        UL_CUDA(c, cudaHostGetDevicePointer((void**)&c->bad_dev, c->bad_host, 0));
    }
    UL_CUDA(c, cudaMemcpyAsync(c->staging_in, host, sizeof(float) * (size_t)n, cudaMemcpyHostToDevice, c->in_stream));
    UL_CUDA(c, cudaEventRecord(c->ev_in_done, c->in_stream));
    c->in_pending = true;
    return UL_OK;
}
int ul_set_links_commit(ul_ctx* c) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    if (!c->in_pending) return fail(c, UL_ESTATE, "no ul_set_links_async to commit");
    DeviceGuard guard(c);
    const long long n = 4 * c->V;
    c->in_pending = false;
    UL_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_in_done, 0));
    *(volatile int*)c->bad_host = 0;                                // nothing on the device writes it before the launch below
    ulk::k_repack<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(geom(c), c->th, c->staging_in, 1, c->bad_dev);
    UL_CUDA(c, cudaGetLastError());
    c->launches += 1;
    UL_CUDA(c, cudaStreamSynchronize(c->stream));
    const int bad = *(volatile int*)c->bad_host;
    if (bad) return fail(c, UL_EINVAL, "link angles must be finite with |theta| <= 3.2 (wrap them to [-pi, pi] first)");
    return UL_OK;
}
int ul_set_links(ul_ctx* c, const float* host) { return links_in(c, host, 1); }
int ul_get_links(ul_ctx* c, float* host) { return links_out(c, host, 0); }
int ul_set_links_raw(ul_ctx* c, const int32_t* host) { return links_in(c, host, 3); }
int ul_get_links_raw(ul_ctx* c, int32_t* host) { return links_out(c, host, 2); }
int ul_get_counter(ul_ctx* c, uint64_t* v) { if (!c || !v) return fail(c, UL_EINVAL, "null pointer"); *v = c->sweep; return UL_OK; }
int ul_set_counter(ul_ctx* c, uint64_t v) { if (!c) return fail(c, UL_EINVAL, "null handle"); c->sweep = v; c->d_sweep_stale = true; return UL_OK; }

int ul_sweep(ul_ctx* c, int n_hb, int n_or) {
    if (!c || n_hb < 0 || n_or < 0) return fail(c, UL_EINVAL, "n_hb, n_or must be >= 0");
    DeviceGuard guard(c);
    NvtxRange range("ul_sweep");
    return compound(c, n_hb, n_or, 0);
}
int ul_substep(ul_ctx* c, int kind, int parity, int mu, int slab_d) {
    if (!c || kind < 0 || kind > 2 || (parity != 0 && parity != 1) || mu < 0 || mu > 3 || slab_d < 0)
        return fail(c, UL_EINVAL, "bad sub-step arguments");
    DeviceGuard guard(c);
    if (slab_d > 0 && c->Nt % slab_d != 0) return fail(c, UL_EINVAL, "Nt % slab_d != 0");
    return substep(c, kind, parity, mu, slab_d);
}
int ul_substep_slabs(ul_ctx* c, int kind, int parity, int mu, int slab_d, int s_begin, int s_end) {
    if (!c || kind < 0 || kind > 2 || (parity != 0 && parity != 1) || mu < 0 || mu > 3 || slab_d < 1 || c->Nt % slab_d != 0)
        return fail(c, UL_EINVAL, "bad sub-step arguments");
    DeviceGuard guard(c);
    if (s_begin < 0 || s_begin > s_end || s_end > c->Nt / slab_d) return fail(c, UL_EINVAL, "bad slab range");
    return substep(c, kind, parity, mu, slab_d, s_begin, s_end);
}
int ul_set_slab_group(ul_ctx* c, int n_slabs) {
    if (!c || n_slabs < -1) return fail(c, UL_EINVAL, "n_slabs must be >= -1");
    if (c->open) return fail(c, UL_ESTATE, "a measurement is open");
    c->slab_group = n_slabs;
    return UL_OK;
}
int ul_set_slab_group_streams(ul_ctx* c, int n_streams) {
    if (!c || n_streams < 1 || n_streams > 8) return fail(c, UL_EINVAL, "n_streams must be 1..8");
    if (c->open) return fail(c, UL_ESTATE, "a measurement is open");
    c->group_streams_n = n_streams;
    return UL_OK;
}
int ul_set_update_algorithm(ul_ctx* c, int alg, double delta) {
    if (!c || (alg != 0 && alg != 1) || (alg == 1 && !(delta > 0.0 && delta <= 3.14159265358979323846)))
        return fail(c, UL_EINVAL, "alg must be 0 (heatbath) or 1 (Metropolis with 0 < delta <= pi)");
    c->alg = alg;
    if (alg == 1) c->met_delta = delta;
    return UL_OK;
}
int ul_set_multihit(ul_ctx* c, int on) {
    if (!c || (on != 0 && on != 1)) return fail(c, UL_EINVAL, "on must be 0 or 1");
    if (c->open) return fail(c, UL_ESTATE, "a measurement is open");
    c->multihit = on != 0;
    return UL_OK;
}
int ul_set_subupdate(ul_ctx* c, int n_hb, int n_or, int k_sweeps) {
    if (!c || n_hb < 0 || n_or < 0 || k_sweeps < 1) return fail(c, UL_EINVAL, "bad sub-update recipe");
    c->sub_hb = n_hb; c->sub_or = n_or; c->sub_k = k_sweeps;
    return UL_OK;
}

int ul_measure_begin(ul_ctx* c, int d, int r_max, const int* fps, int n_fp) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    DeviceGuard guard(c);
    const int rc = check_meas_args(c, d, r_max, fps, n_fp);
    if (rc) return rc;
    return open_measurement(c, d, 0, r_max, fps, n_fp);
}
int ul_set_accum_batch(ul_ctx* c, int depth) {
    if (!c || depth < 0) return fail(c, UL_EINVAL, "depth must be >= 0");
    c->batch_cap = depth;
    return UL_OK;
}
int ul_accumulate(ul_ctx* c) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    DeviceGuard guard(c);
    if (!c->open) return fail(c, UL_ESTATE, "no open measurement");
    const int rc = accumulate(c);
    if (!rc && c->d_out > 0) c->n_inner_acc += 1;
    return rc;
}
int ul_measure_end(ul_ctx* c) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    DeviceGuard guard(c);
    if (!c->open || c->n_acc == 0 || c->d_out > 0) return fail(c, UL_ESTATE, "nothing accumulated (or a two-level measurement is open)");
    const int rc = flush(c);
    if (rc) return rc;
    const double inv = 1.0 / (double)c->n_acc;
    return finish(c, wsp<double2>(c, c->ws.A2), wsp<double2>(c, c->ws.B2), c->n_slab, inv, inv);
}

int ul_multilevel(ul_ctx* c, int d, int n_sub, int r_max, const int* fps, int n_fp) {
    if (!c || n_sub < 0) return fail(c, UL_EINVAL, "n_sub must be >= 0");
    DeviceGuard guard(c);
    NvtxRange range("ul_multilevel");
    int rc = ul_measure_begin(c, d, r_max, fps, n_fp);
    if (rc) return rc;
    auto bail = [&](int code) { c->open = false; return code; };
    if (n_sub == 0) { rc = accumulate(c); if (rc) return bail(rc); }
    const int grp = slab_group_size(c, d);
    if (n_sub > 0 && grp > 0 && grp < c->n_slab) {
        // Slab-group-major order (while the boundary layers are frozen the slabs are dynamically independent): the
        // whole n_sub loop -- masked sub-updates, tables, accumulation -- runs for one group of slabs, whose links and
        // tables stay in L2, before the next group is touched.  Same Philox counters (the sweep counter restarts for
        // every group), same per-entry order of additions: links, counter, slab sums and correlators are bit-identical
        // to the sub-update-major order.
        const uint64_t sweep0 = c->sweep;
        int S = c->group_streams_n;
        if (S > 1 && (c->capturing || group_streams(c, S) != UL_OK)) S = 1;
        for (int g0 = 0; g0 < c->n_slab; g0 += grp * S) {             // a round: S groups side by side, each on its own stream
            const int g1 = g0 + grp * S < c->n_slab ? g0 + grp * S : c->n_slab;
            c->sweep = sweep0; c->d_sweep_stale = true;
            if (S > 1)                                                 // the round's sweep-counter copies
                for (int k = 0; k < S; ++k)
                    ulk::k_set_sweep<<<1, 1, 0, c->stream>>>(c->grp_sweep[k], (uint32_t)(sweep0 & 0xffffffffu), (uint32_t)(sweep0 >> 32));
            c->acc_fresh = true;
            c->n_pending = 0;
            if (S > 1) {                                               // the whole round is one graph replay
                rc = round_run(c, d, g0, g1, grp, S, n_sub);
                if (rc) return bail(rc);
                continue;
            }
            for (int j = 0; j < n_sub; ++j) {
                for (int k = 0; k < c->sub_k; ++k) { rc = compound_direct(c, c->sub_hb, c->sub_or, d, g0, g1); if (rc) return bail(rc); }
                rc = accumulate(c, g0, g1);                            // the round's tables while its links are still in L2
                if (rc) return bail(rc);
                c->n_pending += 1;
                if (c->n_pending == c->ws.kb || j == n_sub - 1) { rc = flush(c, g0, g1); if (rc) return bail(rc); }
            }
        }
        c->n_pending = 0; c->acc_fresh = false;
        c->n_acc = n_sub;
    } else {
        for (int j = 0; j < n_sub; ++j) {
            for (int k = 0; k < c->sub_k; ++k) { rc = compound(c, c->sub_hb, c->sub_or, d); if (rc) return bail(rc); }
            rc = accumulate(c);
            if (rc) return bail(rc);
        }
    }
    rc = ul_measure_end(c);
    return rc ? bail(rc) : rc;
}

// the field points are a full transverse plane fp = b + Ns c <-> (a, b, c) with one a?  (host array)
bool full_plane(const ul_ctx* c, const int* fps, int n_fp, int* a_out) {
    if (c->Ns > ulk::PLANE_MAX_NS || n_fp != c->Ns * c->Ns) return false;
    for (int fp = 0; fp < n_fp; ++fp)
        if (fps[3 * fp] != fps[0] || fps[3 * fp + 1] != fp % c->Ns || fps[3 * fp + 2] != fp / c->Ns) return false;
    *a_out = fps[0];
    return true;
}
// entries per thread of the transverse-DFT kernels: Ns^2 / ept threads per block, at most 1024 (Ns even: Ns^2 % 4 == 0)
int plane_ept(int N2) { return N2 <= 1024 ? 1 : (N2 <= 2048 ? 2 : 4); }
// one configuration's W T O reduction into the result sums: k_replay_reduce, or the transverse-DFT route for full planes
int reduce_fields(ul_ctx* c, const ulk::ReplayArgs& ra, bool plane, int plane_a, int n_entries, double scale) {
    double* res = wsp<double>(c, c->ws.result);
    const long long n = (long long)c->n_slab * c->Vs;
    int nb;
    if (plane) {
        // full transverse plane: DFT route (k_plane_*), results go to Ghat and are transformed back once per measurement
        const int N2 = c->Ns * c->Ns, R = ra.r_max, n_planes = c->n_slab * c->Ns;
        int groups = (148 + R - 1) / R;
        groups = groups > n_planes ? n_planes : groups;
        const size_t oh_b = (size_t)12 * n_planes * N2 * 16, ghp_b = (size_t)groups * R * 12 * N2 * 16, gh_b = (size_t)R * 12 * N2 * 16;
        const size_t need = align_up(oh_b) + align_up(ghp_b) + align_up(gh_b);
        if (need > c->plane_bytes) {
            UL_CUDA(c, cudaStreamSynchronize(c->stream));
            if (c->plane_buf) cudaFree(c->plane_buf);
            c->plane_buf = nullptr; c->plane_bytes = 0;
            void* pb = nullptr;
            UL_CUDA(c, cudaMalloc(&pb, need));
            c->plane_buf = (char*)pb; c->plane_bytes = need;
            c->plane_fresh = true;
        }
        double2* Oh = (double2*)c->plane_buf;
        double2* Ghp = (double2*)(c->plane_buf + align_up(oh_b));
        double2* Gh = (double2*)(c->plane_buf + align_up(oh_b) + align_up(ghp_b));
        if (c->plane_fresh) { UL_CUDA(c, cudaMemsetAsync(Gh, 0, gh_b, c->stream)); c->plane_fresh = false; }
        c->plane_scale = scale; c->plane_r_max = R;
        const size_t smem = (size_t)3 * N2 * sizeof(double2);
        if (!c->plane_attr_set) {
            const int cap = 3 * ulk::PLANE_MAX_NS * ulk::PLANE_MAX_NS * (int)sizeof(double2);
            cudaFuncSetAttribute(ulk::k_plane_dft_o<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
            cudaFuncSetAttribute(ulk::k_plane_dft_o<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
            cudaFuncSetAttribute(ulk::k_plane_dft_o<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
            cudaFuncSetAttribute(ulk::k_plane_spectral<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
            cudaFuncSetAttribute(ulk::k_plane_spectral<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
            cudaFuncSetAttribute(ulk::k_plane_spectral<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
            cudaFuncSetAttribute(ulk::k_plane_idft<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
            cudaFuncSetAttribute(ulk::k_plane_idft<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
            cudaFuncSetAttribute(ulk::k_plane_idft<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
            c->plane_attr_set = true;
        }
        const long long ne = (long long)R * 12 * N2;
        const int ept = plane_ept(N2);                                   // entries per thread: Ns^2 / ept <= 1024 threads
        for (int mu = 1; mu <= 3; ++mu) {
            if (ept == 1) {
                ulk::k_plane_dft_o<1><<<dim3(n_planes, 12), N2, smem, c->stream>>>(ra, mu, Oh);
                ulk::k_plane_spectral<1><<<dim3(R, groups, 2), N2, smem, c->stream>>>(ra, mu, plane_a, Oh, Ghp);
            } else if (ept == 2) {
                ulk::k_plane_dft_o<2><<<dim3(n_planes, 12), N2 / 2, smem, c->stream>>>(ra, mu, Oh);
                ulk::k_plane_spectral<2><<<dim3(R, groups, 4), N2 / 2, smem, c->stream>>>(ra, mu, plane_a, Oh, Ghp);
            } else {
                ulk::k_plane_dft_o<4><<<dim3(n_planes, 12), N2 / 4, smem, c->stream>>>(ra, mu, Oh);
                ulk::k_plane_spectral<4><<<dim3(R, groups, 12), N2 / 4, smem, c->stream>>>(ra, mu, plane_a, Oh, Ghp);
            }
            ulk::k_plane_gh_accum<<<(unsigned)((ne + 255) / 256), 256, 0, c->stream>>>(Ghp, groups, ne, Gh);
        }
        c->launches += 9;
        return cudaGetLastError() == cudaSuccess ? UL_OK : fail(c, UL_ECUDA, "plane reduction launch");
    } else {
        nb = replay_blocks(n);
        ulk::k_replay_reduce<<<dim3(nb, ra.r_max * ra.n_fp), 256, 0, c->stream>>>(ra);
    }
    ulk::k_sum_partials<<<2 * (n_entries - ra.r_max), 256, 0, c->stream>>>(ra.partial + (size_t)2 * ra.r_max * nb, nb, res + 2 * ra.r_max, scale, 1);
    c->launches += 2;
    return cudaGetLastError() == cudaSuccess ? UL_OK : fail(c, UL_ECUDA, "field reduction launch");
}

// Ghat -> the field map in the result buffer (once per measurement, before finish())
int plane_finish(ul_ctx* c, int r_max) {
    const int N2 = c->Ns * c->Ns, n_planes = c->n_slab * c->Ns;
    int groups = (148 + r_max - 1) / r_max;
    groups = groups > n_planes ? n_planes : groups;
    const size_t oh_b = (size_t)12 * n_planes * N2 * 16, ghp_b = (size_t)groups * r_max * 12 * N2 * 16;
    const double2* Gh = (const double2*)(c->plane_buf + align_up(oh_b) + align_up(ghp_b));
    double2* field = (double2*)(wsp<double>(c, c->ws.result) + 2 * r_max);
    const size_t smem = (size_t)3 * N2 * sizeof(double2);
    const int ept = plane_ept(N2);
    if (ept == 1) ulk::k_plane_idft<1><<<dim3(r_max, 12), N2, smem, c->stream>>>(Gh, c->Ns, c->plane_scale, field);
    else if (ept == 2) ulk::k_plane_idft<2><<<dim3(r_max, 12), N2 / 2, smem, c->stream>>>(Gh, c->Ns, c->plane_scale, field);
    else ulk::k_plane_idft<4><<<dim3(r_max, 12), N2 / 4, smem, c->stream>>>(Gh, c->Ns, c->plane_scale, field);
    c->launches += 1;
    c->plane_fresh = true;
    return cudaGetLastError() == cudaSuccess ? UL_OK : fail(c, UL_ECUDA, "k_plane_idft launch");
}

// Single-level measurement by replay: the same estimator, trajectory and results as
// ul_multilevel (to fp64 rounding order), with 2x the sweeps and none of the per-site TO accumulators.
int ul_multilevel_replay(ul_ctx* c, int d, int n_sub, int r_max, const int* fps, int n_fp) {
    if (!c || n_sub < 0) return fail(c, UL_EINVAL, "n_sub must be >= 0");
    DeviceGuard guard(c);
    if (n_fp == 0) return ul_multilevel(c, d, n_sub, r_max, fps, n_fp);                  // nothing is linear in O: nothing to replay
    int rc = check_meas_args(c, d, r_max, fps, n_fp);
    if (rc) return rc;
    int plane_a = 0;
    const bool plane = full_plane(c, fps, n_fp, &plane_a);
    rc = ensure_staging(c);
    if (rc) return rc;
    const size_t link_bytes = sizeof(float) * 4 * (size_t)c->V;
    UL_CUDA(c, cudaMemcpyAsync(c->staging, c->th, link_bytes, cudaMemcpyDeviceToDevice, c->stream));   // start configuration
    const uint64_t sweep0 = c->sweep;
    c->replay = true;
    rc = open_measurement(c, d, 0, r_max, fps, n_fp);
    if (rc) { c->replay = false; return rc; }
    auto bail = [&](int code) { c->replay = false; c->open = false; return code; };
    // pass 1: sums of T only
    if (n_sub == 0) { rc = accumulate(c); if (rc) return bail(rc); }
    for (int j = 0; j < n_sub; ++j) {
        for (int k = 0; k < c->sub_k; ++k) { rc = compound(c, c->sub_hb, c->sub_or, d); if (rc) return bail(rc); }
        rc = accumulate(c);
        if (rc) return bail(rc);
    }
    rc = flush(c);
    if (rc) return bail(rc);
    const double inv = 1.0 / (double)c->n_acc;
    ulk::WeightArgs wa;
    wa.Vs = c->Vs; wa.r_max = r_max; wa.n_slab = c->n_slab; wa.inv = inv;
    wa.A = wsp<double2>(c, c->ws.A2); wa.W = wsp<double2>(c, c->ws.B2);
    const long long nw = 3LL * r_max * c->Vs;
    ulk::k_slab_weights<<<(unsigned)((nw + 255) / 256), 256, 0, c->stream>>>(wa);
    if (cudaGetLastError() != cudaSuccess) return bail(fail(c, UL_ECUDA, "k_slab_weights launch"));
    c->launches += 1;
    // pass 2: the same trajectory again, fields reduced on the fly
    if (n_sub > 0) {
        if (cudaMemcpyAsync(c->th, c->staging, link_bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return bail(fail(c, UL_ECUDA, "restore links"));
        c->sweep = sweep0;
        c->d_sweep_stale = true;
    }
    const long long n = (long long)c->n_slab * c->Vs;
    const int n_entries = r_max * (1 + 12 * n_fp);
    double* res = wsp<double>(c, c->ws.result);
    ulk::TableArgs t;
    t.g = geom(c); t.th = c->th; t.d = c->d; t.n_slab = c->n_slab;
    t.U = wsp<double2>(c, c->ws.U); t.Um = nullptr; t.beta = (float)c->beta;       // the TO sums use the plain T
    t.Ot = wsp<float>(c, c->ws.Ot); t.partial = wsp<double>(c, c->ws.partial);
    t.row0 = 0; t.n_rows = c->n_slab * c->Ns;
    ulk::ReplayArgs ra;
    ra.g = geom(c); ra.n_slab = c->n_slab; ra.r_max = r_max; ra.n_fp = n_fp;
    ra.U = t.U; ra.Ot = t.Ot; ra.fps = wsp<int>(c, c->ws.fps); ra.W = wa.W; ra.partial = wsp<double>(c, c->ws.partial);
    const int gx = (c->Ns * c->Ns + 255) / 256, rows = c->n_slab * c->Ns;
    const int gy = rows < TBLK / gx ? rows : (TBLK / gx > 0 ? TBLK / gx : 1);
    const int nb = replay_blocks(n);
    const double scale = inv / (3.0 * (double)c->Vs * (double)c->Nt);                    // Eq. 34 normalisation and 1/n_sub
    for (int j = 0; j < (n_sub > 0 ? n_sub : 1); ++j) {
        if (n_sub > 0)
            for (int k = 0; k < c->sub_k; ++k) { rc = compound(c, c->sub_hb, c->sub_or, d); if (rc) return bail(rc); }
        ulk::k_slab_tables<<<dim3(gx, gy), 256, 0, c->stream>>>(t);                      // column sums were taken in pass 1
        c->launches += 1;
        rc = reduce_fields(c, ra, plane, plane_a, n_entries, scale);
        if (rc) return bail(rc);
    }
    if (plane) { rc = plane_finish(c, r_max); if (rc) return bail(rc); }
    rc = finish(c, wsp<double2>(c, c->ws.A2), nullptr, c->n_slab, inv, inv);
    c->replay = false;
    return rc;
}

// Two levels (S8(c)-O7), Alg. 1 lines 5 / 16 / 18 as three steps shared by ul_multilevel2 and the test hooks
// ul_measure2_begin / ul_combine / ul_measure2_end.
static int begin2(ul_ctx* c, int d_in, int d_out, int r_max, const int* fps, int n_fp) {
    int rc = check_meas_args(c, d_in, r_max, fps, n_fp);
    if (rc) return rc;
    if (d_out < d_in || d_out % d_in != 0 || c->Nt % d_out != 0) return fail(c, UL_EINVAL, "need d_in | d_out | Nt");
    rc = open_measurement(c, d_in, d_out, r_max, fps, n_fp);
    if (rc) return rc;
    c->n_comb = 0; c->n_in_seen = 0; c->n_inner_acc = 0;
    return UL_OK;
}
// Eqs. 32-33 on the inner averages (inner sums / number of configurations accumulated since the last combine),
// added to the outer sums; the next inner sums start from zero
static int combine2(ul_ctx* c) {
    if (c->n_inner_acc < 1) return fail(c, UL_ESTATE, "nothing accumulated since the last combine");
    if (c->n_comb > 0 && c->n_inner_acc != c->n_in_seen) return fail(c, UL_ESTATE, "every outer iteration must accumulate the same number of configurations");
    const int rc = flush(c);
    if (rc) return rc;
    const Workspace& w = c->ws;
    ulk::CombineArgs a;
    a.Vs = c->Vs; a.r_max = c->r_max; a.n_fp = c->n_fp; a.n_inner = c->n_slab; a.n_outer = c->n_outer; a.m = c->d_out / c->d;
    a.inv = 1.0 / (double)c->n_inner_acc;
    a.A2 = wsp<double2>(c, w.A2); a.B2 = wsp<double2>(c, w.B2); a.A4 = wsp<double2>(c, w.A4); a.B4 = wsp<double2>(c, w.B4);
    const long long total = 3LL * c->r_max * c->n_outer * c->Vs;
    ulk::k_combine<<<(unsigned)((total + 255) / 256), 256, 0, c->stream>>>(a);
    UL_CUDA(c, cudaGetLastError());
    c->launches += 1;
    c->n_in_seen = c->n_inner_acc;
    c->n_inner_acc = 0;
    c->n_comb += 1;
    c->acc_fresh = true;                                                                     // A2, B2 <- 0
    return UL_OK;
}
static int end2(ul_ctx* c) {
    if (c->n_comb < 1 || c->n_inner_acc != 0) return fail(c, UL_ESTATE, "nothing combined, or configurations accumulated since the last combine");
    const Workspace& w = c->ws;
    return finish(c, wsp<double2>(c, w.A4), wsp<double2>(c, w.B4), c->n_outer, 1.0 / (double)c->n_comb,
                  1.0 / ((double)c->n_in_seen * (double)c->n_comb));
}
int ul_multilevel2(ul_ctx* c, int d_in, int n_in, int d_out, int n_out, int r_max, const int* fps, int n_fp) {
    if (!c || n_in < 1 || n_out < 1) return fail(c, UL_EINVAL, "n_in, n_out must be >= 1");
    DeviceGuard guard(c);
    int rc = begin2(c, d_in, d_out, r_max, fps, n_fp);
    if (rc) return rc;
    auto bail = [&](int code) { c->open = false; return code; };
    for (int J = 0; J < n_out; ++J) {
        for (int k = 0; k < c->sub_k; ++k) { rc = compound(c, c->sub_hb, c->sub_or, d_out); if (rc) return bail(rc); }
        for (int j = 0; j < n_in; ++j) {
            for (int k = 0; k < c->sub_k; ++k) { rc = compound(c, c->sub_hb, c->sub_or, d_in); if (rc) return bail(rc); }
            rc = accumulate(c);
            if (rc) return bail(rc);
            c->n_inner_acc += 1;
        }
        rc = combine2(c);
        if (rc) return bail(rc);
    }
    rc = end2(c);
    return rc ? bail(rc) : rc;
}
int ul_measure2_begin(ul_ctx* c, int d_in, int d_out, int r_max, const int* fps, int n_fp) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    DeviceGuard guard(c);
    return begin2(c, d_in, d_out, r_max, fps, n_fp);
}
int ul_combine(ul_ctx* c) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    DeviceGuard guard(c);
    if (!c->open || c->d_out == 0) return fail(c, UL_ESTATE, "no open two-level measurement");
    return combine2(c);
}
int ul_measure2_end(ul_ctx* c) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    DeviceGuard guard(c);
    if (!c->open || c->d_out == 0) return fail(c, UL_ESTATE, "no open two-level measurement");
    return end2(c);
}

// Two levels by replay (S8(f) rank 2 for BJ config 4): G is linear in O, with weights that need the inner averages of
// the same outer iteration and the outer averages of the whole measurement.  Pass 1 runs the two-level measurement with
// the sums of T only (-> [T4], C(r), W4).  Pass 2 restarts from the saved configuration; in every outer iteration the
// inner loop is run twice from a saved configuration: once to form [T2] and the combined weights Wc, once to reduce
// Wc T2 O on the fly.  About three times the sub-update sweeps of ul_multilevel2, none of its TO accumulators.
int ul_multilevel2_replay(ul_ctx* c, int d_in, int n_in, int d_out, int n_out, int r_max, const int* fps, int n_fp) {
    if (!c || n_in < 1 || n_out < 1) return fail(c, UL_EINVAL, "n_in, n_out must be >= 1");
    DeviceGuard guard(c);
    if (n_fp == 0) return ul_multilevel2(c, d_in, n_in, d_out, n_out, r_max, fps, n_fp);
    int rc = check_meas_args(c, d_in, r_max, fps, n_fp);
    if (rc) return rc;
    int plane_a = 0;
    const bool plane = full_plane(c, fps, n_fp, &plane_a);
    if (d_out < d_in || d_out % d_in != 0 || c->Nt % d_out != 0) return fail(c, UL_EINVAL, "need d_in | d_out | Nt");
    rc = ensure_staging(c);
    if (rc) return rc;
    const size_t link_bytes = sizeof(float) * 4 * (size_t)c->V;
    if (!c->staging2) { void* p = nullptr; UL_CUDA(c, cudaMalloc(&p, link_bytes)); c->staging2 = (float*)p; }
    UL_CUDA(c, cudaMemcpyAsync(c->staging, c->th, link_bytes, cudaMemcpyDeviceToDevice, c->stream));
    const uint64_t sweep0 = c->sweep;
    c->replay = true;
    rc = open_measurement(c, d_in, d_out, r_max, fps, n_fp);
    if (rc) { c->replay = false; return rc; }
    auto bail = [&](int code) { c->replay = false; c->skip_colsum = false; c->open = false; return code; };
    const Workspace& w = c->ws;
    ulk::CombineArgs ca;
    ca.Vs = c->Vs; ca.r_max = r_max; ca.n_fp = 0; ca.n_inner = c->n_slab; ca.n_outer = c->n_outer; ca.m = d_out / d_in;
    ca.inv = 1.0 / (double)n_in;
    ca.A2 = wsp<double2>(c, w.A2); ca.B2 = nullptr; ca.A4 = wsp<double2>(c, w.A4); ca.B4 = nullptr;
    const long long total = 3LL * r_max * c->n_outer * c->Vs;
    auto inner_pass = [&]() {                                      // n_in inner sub-updates, sums of T into A2
        c->acc_fresh = true;
        for (int j = 0; j < n_in; ++j) {
            for (int k = 0; k < c->sub_k; ++k) { const int e = compound(c, c->sub_hb, c->sub_or, d_in); if (e) return e; }
            const int e = accumulate(c);
            if (e) return e;
        }
        return flush(c);
    };
    // pass 1
    for (int J = 0; J < n_out; ++J) {
        for (int k = 0; k < c->sub_k; ++k) { rc = compound(c, c->sub_hb, c->sub_or, d_out); if (rc) return bail(rc); }
        rc = inner_pass();
        if (rc) return bail(rc);
        ulk::k_combine<<<(unsigned)((total + 255) / 256), 256, 0, c->stream>>>(ca);
        c->launches += 1;
    }
    ulk::WeightArgs wa;
    wa.Vs = c->Vs; wa.r_max = r_max; wa.n_slab = c->n_outer; wa.inv = 1.0 / (double)n_out;
    wa.A = ca.A4; wa.W = wsp<double2>(c, w.B4);                    // W4 in the (A4-sized) B4 slot
    const long long nw = 3LL * r_max * c->Vs;
    ulk::k_slab_weights<<<(unsigned)((nw + 255) / 256), 256, 0, c->stream>>>(wa);
    c->launches += 1;
    if (cudaGetLastError() != cudaSuccess) return bail(fail(c, UL_ECUDA, "two-level replay, pass 1"));
    // pass 2
    if (cudaMemcpyAsync(c->th, c->staging, link_bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return bail(fail(c, UL_ECUDA, "restore links"));
    c->sweep = sweep0; c->d_sweep_stale = true;
    c->skip_colsum = true;
    const long long n = (long long)c->n_slab * c->Vs;
    const int n_entries = r_max * (1 + 12 * n_fp);
    double* res = wsp<double>(c, w.result);
    ulk::GroupWeightArgs ga;
    ga.Vs = c->Vs; ga.r_max = r_max; ga.n_inner = c->n_slab; ga.n_outer = c->n_outer; ga.m = d_out / d_in; ga.inv = 1.0 / (double)n_in;
    ga.A2 = ca.A2; ga.W4 = wa.W; ga.Wc = wsp<double2>(c, w.B2);    // Wc in the (A2-sized) B2 slot
    ulk::TableArgs t;
    t.g = geom(c); t.th = c->th; t.d = c->d; t.n_slab = c->n_slab;
    t.U = wsp<double2>(c, w.U); t.Um = nullptr; t.beta = (float)c->beta;
    t.Ot = wsp<float>(c, w.Ot); t.partial = wsp<double>(c, w.partial);
    t.row0 = 0; t.n_rows = c->n_slab * c->Ns;
    ulk::ReplayArgs ra;
    ra.g = geom(c); ra.n_slab = c->n_slab; ra.r_max = r_max; ra.n_fp = n_fp;
    ra.U = t.U; ra.Ot = t.Ot; ra.fps = wsp<int>(c, w.fps); ra.W = ga.Wc; ra.partial = wsp<double>(c, w.partial);
    const int gx = (c->Ns * c->Ns + 255) / 256, rows = c->n_slab * c->Ns;
    const int gy = rows < TBLK / gx ? rows : (TBLK / gx > 0 ? TBLK / gx : 1);
    const int nb = replay_blocks(n);
    const double scale = 1.0 / ((double)n_in * (double)n_out * 3.0 * (double)c->Vs * (double)c->Nt);
    for (int J = 0; J < n_out; ++J) {
        for (int k = 0; k < c->sub_k; ++k) { rc = compound(c, c->sub_hb, c->sub_or, d_out); if (rc) return bail(rc); }
        if (cudaMemcpyAsync(c->staging2, c->th, link_bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return bail(fail(c, UL_ECUDA, "save links"));
        const uint64_t sweepJ = c->sweep;
        rc = inner_pass();                                         // (a) the inner averages of this outer iteration
        if (rc) return bail(rc);
        ulk::k_group_weights<<<(unsigned)((nw + 255) / 256), 256, 0, c->stream>>>(ga);
        c->launches += 1;
        if (cudaMemcpyAsync(c->th, c->staging2, link_bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return bail(fail(c, UL_ECUDA, "restore links"));
        c->sweep = sweepJ; c->d_sweep_stale = true;
        for (int j = 0; j < n_in; ++j) {                           // (b) the same inner sub-updates again, fields reduced on the fly
            for (int k = 0; k < c->sub_k; ++k) { rc = compound(c, c->sub_hb, c->sub_or, d_in); if (rc) return bail(rc); }
            ulk::k_slab_tables<<<dim3(gx, gy), 256, 0, c->stream>>>(t);
            c->launches += 1;
            rc = reduce_fields(c, ra, plane, plane_a, n_entries, scale);
            if (rc) return bail(rc);
        }
        if (cudaGetLastError() != cudaSuccess) return bail(fail(c, UL_ECUDA, "two-level replay, pass 2"));
    }
    c->skip_colsum = false;
    if (plane) { rc = plane_finish(c, r_max); if (rc) return bail(rc); }
    rc = finish(c, ca.A4, nullptr, c->n_outer, 1.0 / (double)n_out, 1.0 / ((double)n_in * (double)n_out));
    c->replay = false;
    return rc;
}

int ul_plaquette(ul_ctx* c, double* out) {
    if (!c || !out) return fail(c, UL_EINVAL, "null pointer");
    DeviceGuard guard(c);
    const int gx = (c->Ns * c->Ns + 255) / 256, rows = c->Nt * c->Ns;
    const int gy = rows < NBLK / gx ? rows : (NBLK / gx > 0 ? NBLK / gx : 1);
    if (gx * gy > NBLK) return fail(c, UL_EINVAL, "lattice too large for this build");
    ulk::k_plaquette<<<dim3(gx, gy), 256, 0, c->stream>>>(geom(c), c->th, c->scratch);
    ulk::k_sum_partials<<<2, 256, 0, c->stream>>>(c->scratch, gx * gy, c->scratch + 2 * NBLK, 1.0 / (3.0 * (double)c->V), 0);
    UL_CUDA(c, cudaGetLastError());
    c->launches += 2;
    double v[2];
    UL_CUDA(c, cudaMemcpyAsync(v, c->scratch + 2 * NBLK, sizeof(v), cudaMemcpyDeviceToHost, c->stream));
    UL_CUDA(c, cudaStreamSynchronize(c->stream));
    out[0] = 0.5 * (v[0] + v[1]); out[1] = v[0]; out[2] = v[1];
    return UL_OK;
}
// ---- the plaquette average without any allocation (include/ul.h: ul_plaquette_noalloc) -------------------------------------
// The block partials and the two sums of k_plaquette / k_sum_partials live in a file-scope device array instead of the
// cudaMalloc'ed scratch of the handle: 2 NBLK + 4 doubles = 9.5 KB, held by every GPU that loads the library until it exits.
// In host code the NAME of the array is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, taken once per device with that device current (device code of this file could name the array directly).
static __device__ __align__(256) double g_plaq_scratch[2 * NBLK + 4];
static double* g_plaq_scratch_ptr[64] = {};                        // per device, resolved on the first call for that device

// (mean over all, time-like, space-like) from the two sums; out = caller's device buffer
static __global__ void k_plaquette_out(const double* __restrict__ sums, double* __restrict__ out) {
    if (threadIdx.x == 0) { const double t = sums[0], sp = sums[1]; out[0] = 0.5 * (t + sp); out[1] = t; out[2] = sp; }
}

int ul_plaquette_noalloc(ul_ctx* c, double* dev_out) {
    if (!c || !dev_out) return fail(c, UL_EINVAL, "null pointer");
    if (c->dev < 0 || c->dev >= 64) return fail(c, UL_EINVAL, "ul_plaquette_noalloc: device index beyond 63");
    // the fixed scratch holds one partial per block and sum, at most NBLK blocks: ceil(Ns^2 / 256) <= NBLK, i.e. Ns <= 389
    const int gx = (c->Ns * c->Ns + 255) / 256, rows = c->Nt * c->Ns;
    if (gx > NBLK)
        return fail(c, UL_EINVAL, "ul_plaquette_noalloc: lattice beyond the fixed scratch (need ceil(Ns^2 / 256) <= 592 blocks, i.e. Ns <= 389)");
    const int gy = rows < NBLK / gx ? rows : NBLK / gx;             // gx gy <= NBLK
    DeviceGuard guard(c);                                            // the context's device is current from here on
    double* scratch = g_plaq_scratch_ptr[c->dev];
    if (!scratch) {                                                  // set-up, once per device: no allocation, a symbol lookup
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_plaq_scratch);
        if (e != cudaSuccess || !p) return fail(c, UL_ECUDA, std::string("cudaGetSymbolAddress(g_plaq_scratch): ") + cudaGetErrorString(e));
        scratch = g_plaq_scratch_ptr[c->dev] = (double*)p;
    }
    // every element read below is written by this call first (gx gy partials per sum, then the two sums), so nothing has to
    // start at zero although the array keeps the last call's contents
    ulk::k_plaquette<<<dim3(gx, gy), 256, 0, c->stream>>>(geom(c), c->th, scratch);
    ulk::k_sum_partials<<<2, 256, 0, c->stream>>>(scratch, gx * gy, scratch + 2 * NBLK, 1.0 / (3.0 * (double)c->V), 0);
    k_plaquette_out<<<1, 32, 0, c->stream>>>(scratch + 2 * NBLK, dev_out);
    UL_CUDA(c, cudaGetLastError());
    c->launches += 3;
    return UL_OK;
}
int ul_polyakov(ul_ctx* c, int multihit, double* out) {
    if (!c || !out || (multihit != 0 && multihit != 1)) return fail(c, UL_EINVAL, "multihit must be 0 or 1");
    DeviceGuard guard(c);
    const int nb = (int)((c->Vs + 255) / 256) < NBLK ? (int)((c->Vs + 255) / 256) : NBLK;
    ulk::k_polyakov<<<nb, 256, 0, c->stream>>>(geom(c), c->th, c->beta, multihit, c->scratch);
    ulk::k_sum_partials<<<2, 256, 0, c->stream>>>(c->scratch, nb, c->scratch + 2 * NBLK, 1.0 / (double)c->Vs, 0);
    UL_CUDA(c, cudaGetLastError());
    c->launches += 2;
    UL_CUDA(c, cudaMemcpyAsync(out, c->scratch + 2 * NBLK, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    UL_CUDA(c, cudaStreamSynchronize(c->stream));
    return UL_OK;
}
int ul_read_correlators(ul_ctx* c, double* corr, double* field, double* vacuum) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    if (!c->have) return fail(c, UL_ESTATE, "no measurement yet");
    if (corr) std::memcpy(corr, c->corr.data(), sizeof(double) * c->corr.size());
    if (field && !c->field.empty()) std::memcpy(field, c->field.data(), sizeof(double) * c->field.size());
    if (vacuum) std::memcpy(vacuum, c->vacuum.data(), sizeof(double) * 12);
    return UL_OK;
}
int ul_read_slab_averages(ul_ctx* c, double* out) {
    if (!c || !out) return fail(c, UL_EINVAL, "null pointer");
    DeviceGuard guard(c);
    if (!c->have) return fail(c, UL_ESTATE, "no measurement yet");
    const size_t n = (size_t)3 * c->res_r_max * c->res_n_slab * (size_t)c->Vs * 2;
    UL_CUDA(c, cudaMemcpyAsync(out, c->res_A, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
    UL_CUDA(c, cudaStreamSynchronize(c->stream));
    for (size_t i = 0; i < n; ++i) out[i] *= c->res_inv;
    return UL_OK;
}
int ul_set_site_offset(ul_ctx* c, int64_t offset) {
    if (!c || offset < -(int64_t)c->V || offset + (int64_t)c->V > ((int64_t)1 << 29))
        return fail(c, UL_EINVAL, "need -V <= site offset and site offset + local volume <= 2^29");
    c->site_offset = (uint32_t)(uint64_t)offset;      // mod 2^32: a negative offset (ghost layers below t0) wraps back for the own layers
    return UL_OK;
}
int ul_slab_partial_product(ul_ctx* c, int s_begin, int s_end, void* dev_out) {
    if (!c || !dev_out) return fail(c, UL_EINVAL, "null pointer");
    DeviceGuard guard(c);
    if (!c->have) return fail(c, UL_ESTATE, "no measurement yet");
    if (s_begin < 0 || s_end > c->res_n_slab || s_begin > s_end) return fail(c, UL_EINVAL, "bad slab range");
    ulk::WeightArgs wa;
    wa.Vs = c->Vs; wa.r_max = c->res_r_max; wa.n_slab = c->res_n_slab; wa.inv = c->res_inv;
    wa.A = c->res_A; wa.W = (double2*)dev_out;
    const long long nw = 3LL * wa.r_max * c->Vs;
    ulk::k_slab_partial_product<<<(unsigned)((nw + 255) / 256), 256, 0, c->stream>>>(wa, s_begin, s_end);
    UL_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return UL_OK;
}
int ul_combine_partial_products(ul_ctx* c, const void* const* dev_parts, int n_parts, double* corr) {
    if (!c || !dev_parts || !corr) return fail(c, UL_EINVAL, "null pointer");
    DeviceGuard guard(c);
    if (n_parts < 1 || n_parts > ulk::MAX_SHARDS) return fail(c, UL_EINVAL, "need 1 <= n_parts <= 64");
    if (!c->have) return fail(c, UL_ESTATE, "no measurement yet");
    ulk::CombinePartsArgs a;
    a.Vs = c->Vs; a.r_max = c->res_r_max; a.n_parts = n_parts;
    for (int k = 0; k < n_parts; ++k) {
        if (!dev_parts[k]) return fail(c, UL_EINVAL, "null partial product");
        a.part[k] = (const double2*)dev_parts[k];
    }
    a.partial = wsp<double>(c, c->ws.partial);                 // >= 2 r_max NBLK doubles (plan_workspace)
    double* res = wsp<double>(c, c->ws.result);
    const int R = c->res_r_max;
    ulk::k_combine_partial_products<<<dim3(NBLK, R), 256, 0, c->stream>>>(a);
    ulk::k_sum_partials<<<2 * R, 256, 0, c->stream>>>(a.partial, NBLK, res, 1.0 / (3.0 * (double)c->Vs), 0);
    UL_CUDA(c, cudaGetLastError());
    c->launches += 2;
    UL_CUDA(c, cudaMemcpyAsync(corr, res, sizeof(double) * 2 * (size_t)R, cudaMemcpyDeviceToHost, c->stream));
    UL_CUDA(c, cudaStreamSynchronize(c->stream));
    c->corr.assign(corr, corr + 2 * R);                        // ul_read_correlators now returns the global C(r)
    return UL_OK;
}
int ul_set_halo_peers(ul_ctx* c, void* dn_links, void* up_links, int ghost_layers) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    if (c->open) return fail(c, UL_ESTATE, "a measurement is open");
    if (!dn_links && !up_links) { c->peer_dn = c->peer_up = nullptr; c->peer_flag_dn = c->peer_flag_up = nullptr; c->halo_gl = 0; return UL_OK; }
    if (!dn_links || !up_links || ghost_layers < 2 || (ghost_layers & 1) || c->Nt - 2 * ghost_layers < ghost_layers)
        return fail(c, UL_EINVAL, "need both neighbours, an even number >= 2 of ghost layers and at least that many own layers");
    DeviceGuard guard(c);
    for (void* p : {dn_links, up_links}) {                        // a neighbour on another device of this process: enable peer access
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, p) != cudaSuccess || at.type != cudaMemoryTypeDevice) { cudaGetLastError(); return fail(c, UL_EINVAL, "peer links must be device memory"); }
        if (at.device != c->dev) {
            int can = 0;
            cudaDeviceCanAccessPeer(&can, c->dev, at.device);
            if (!can) return fail(c, UL_ECUDA, "no peer access to the neighbour's device");
            const cudaError_t e = cudaDeviceEnablePeerAccess(at.device, 0);
            if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) return fail(c, UL_ECUDA, std::string("cudaDeviceEnablePeerAccess: ") + cudaGetErrorString(e));
            cudaGetLastError();
        }
    }
    c->peer_dn = (int*)dn_links; c->peer_up = (int*)up_links; c->halo_gl = ghost_layers;
    return UL_OK;
}
int ul_halo_flags(ul_ctx* c, void** dev_flags) {
    if (!c || !dev_flags) return fail(c, UL_EINVAL, "null pointer");
    DeviceGuard guard(c);
    if (!c->halo_flags) {
        void* p = nullptr;
        UL_CUDA(c, cudaMalloc(&p, 2 * sizeof(uint32_t)));
        c->halo_flags = (uint32_t*)p;
    }
    UL_CUDA(c, cudaMemsetAsync(c->halo_flags, 0, 2 * sizeof(uint32_t), c->stream));
    UL_CUDA(c, cudaStreamSynchronize(c->stream));
    c->halo_seq = 0;
    *dev_flags = c->halo_flags;
    return UL_OK;
}
int ul_set_halo_peer_flags(ul_ctx* c, void* dn_flags, void* up_flags) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    if (!dn_flags || !up_flags) { c->peer_flag_dn = c->peer_flag_up = nullptr; return UL_OK; }
    if (!c->halo_flags) return fail(c, UL_ESTATE, "call ul_halo_flags first");
    c->peer_flag_dn = (uint32_t*)dn_flags + 1;                    // the shard below hears from its upper neighbour in its flags[1]
    c->peer_flag_up = (uint32_t*)up_flags;                        // the shard above from its lower neighbour in its flags[0]
    c->halo_seq = 0;
    return UL_OK;
}
// ---- the same between PROCESSES (one process per GPU): CUDA IPC handles of the link array and the flag words
int ul_ipc_export(ul_ctx* c, void* out_links_handle, uint64_t* links_offset, void* out_flags_handle, uint64_t* flags_offset) {
    if (!c || !out_links_handle || !links_offset || !out_flags_handle || !flags_offset) return fail(c, UL_EINVAL, "null pointer");
    DeviceGuard guard(c);
    if (!c->halo_flags) return fail(c, UL_ESTATE, "call ul_halo_flags first");
    typedef int (*GetRange)(unsigned long long*, size_t*, unsigned long long);
    static GetRange get_range = [] {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult st;
        return (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &st) == cudaSuccess && st == cudaDriverEntryPointSuccess) ? (GetRange)fn : (GetRange) nullptr;
    }();
    if (!get_range) return fail(c, UL_ECUDA, "cuMemGetAddressRange not available");
    const void* ptrs[2] = {c->th, c->halo_flags};
    void* outs[2] = {out_links_handle, out_flags_handle};
    uint64_t* offs[2] = {links_offset, flags_offset};
    for (int i = 0; i < 2; ++i) {                                 // a handle names the whole allocation: pass the offset inside it along
        unsigned long long base = 0;
        size_t size = 0;
        if (get_range(&base, &size, (unsigned long long)(uintptr_t)ptrs[i]) != 0) return fail(c, UL_ECUDA, "cuMemGetAddressRange");
        cudaIpcMemHandle_t hnd;
        UL_CUDA(c, cudaIpcGetMemHandle(&hnd, (void*)(uintptr_t)base));
        std::memcpy(outs[i], &hnd, sizeof(hnd));
        *offs[i] = (uint64_t)((uintptr_t)ptrs[i] - (uintptr_t)base);
    }
    return UL_OK;
}
int ul_ipc_open(ul_ctx* c, const void* handle, uint64_t offset, void** dev_ptr) {
    if (!c || !handle || !dev_ptr) return fail(c, UL_EINVAL, "null pointer");
    DeviceGuard guard(c);
    cudaIpcMemHandle_t hnd;
    std::memcpy(&hnd, handle, sizeof(hnd));
    for (auto& e : c->ipc_open)                                    // an allocation is opened once per process
        if (std::memcmp(&e.first, &hnd, sizeof(hnd)) == 0) { *dev_ptr = (char*)e.second + offset; return UL_OK; }
    void* base = nullptr;
    UL_CUDA(c, cudaIpcOpenMemHandle(&base, hnd, cudaIpcMemLazyEnablePeerAccess));
    c->ipc_open.push_back({hnd, base});
    *dev_ptr = (char*)base + offset;
    return UL_OK;
}
int ul_get_launch_count(ul_ctx* c, uint64_t* n) { if (!c || !n) return fail(c, UL_EINVAL, "null pointer"); *n = c->launches; return UL_OK; }

int ul_philox_selftest(const uint32_t* ctr, const uint32_t* key, uint32_t* out, int n) {
    if (!ctr || !key || !out || n < 1) return fail(nullptr, UL_EINVAL, "bad arguments");
    uint32_t* d = nullptr;
    UL_CUDA(nullptr, cudaMalloc((void**)&d, sizeof(uint32_t) * 10 * (size_t)n));
    uint32_t *dc = d, *dk = d + 4 * (size_t)n, *dout = d + 6 * (size_t)n;
    cudaError_t e = cudaMemcpy(dc, ctr, sizeof(uint32_t) * 4 * (size_t)n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(dk, key, sizeof(uint32_t) * 2 * (size_t)n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) { ulk::k_philox_test<<<(n + 127) / 128, 128>>>(dc, dk, dout, n); e = cudaGetLastError(); }
    if (e == cudaSuccess) e = cudaMemcpy(out, dout, sizeof(uint32_t) * 4 * (size_t)n, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return fail(nullptr, UL_ECUDA, cudaGetErrorString(e));
    return UL_OK;
}
int ul_sync(ul_ctx* c) {
    if (!c) return fail(c, UL_EINVAL, "null handle");
    DeviceGuard guard(c);
    UL_CUDA(c, cudaStreamSynchronize(c->stream));
    return UL_OK;
}
const char* ul_last_error(ul_ctx* c) { return c ? c->err.c_str() : g_err.c_str(); }

}  // extern "C"
