/* ul.h -- C ABI of libul.so: the B200-native hot path of arXiv:1309.3859
 * (Amado, Cardoso, Bicudo): compact U(1) Wilson-action lattice gauge theory in 3+1 d,
 * heatbath + overrelaxation checkerboard sweeps, slab-masked sub-updates and the
 * Luescher-Weisz multilevel estimator of <P^dagger P> and <P^dagger P O>.
 *
 * Citations: "P:<n>" = line n of the paper text; "S8" = SURVEY.md section 8;
 * "DESIGN R<k>" = reading k in DESIGN.md.
 *
 * Conventions (S8): directions mu = 0 (time), 1,2,3 = x,y,z.  Site index
 * i = x1 + Ns*(x2 + Ns*(x3 + Ns*t)); parity (x1+x2+x3+t) mod 2.  "Canonical" link arrays
 * at this boundary are HOST pointers to float[4][Nt][Ns][Ns][Ns] (mu slowest, x1 fastest),
 * fp32 radians in [-pi, pi].  Inside the library the links live in HBM as 32-bit binary angles
 * (int32 I, theta = I * 2 pi / 2^32: angle sums are exact wrapping adds) in a parity-split,
 * direction-split structure of arrays.  fp32 radians -> binary angle ->
 * fp32 radians returns the same fp32 for |theta| >= 2^-6 rad and differs by <= 1.2e-9 rad
 * below that.
 *
 * Ownership: the library owns the handle.  Every host pointer passed in is caller-owned and
 * only read or written during the call.  With ul_create_ext the caller also owns the device
 * buffers (e.g. torch.empty) and the stream (e.g. torch.cuda.Stream.cuda_stream); they must
 * outlive the handle and the library never frees them.  With ul_create the library
 * cudaMallocs and frees its own buffers and uses its own stream.
 *
 * Errors: every call returns UL_OK (0) or a negative code; nothing aborts or throws.
 * ul_last_error(h) returns a static / handle-owned string describing the last failure.
 * All calls are synchronous with respect to the host unless stated (ul_sweep and the
 * multilevel calls only enqueue on the handle's stream; reads synchronise).
 * There is no CPU fallback: without a CUDA device every call that touches the lattice
 * returns UL_ECUDA.
 */
#ifndef UL_H
#define UL_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ul_ctx ul_ctx;
enum { UL_OK = 0, UL_EINVAL = -1, UL_ENOMEM = -2, UL_ECUDA = -3, UL_ESTATE = -4 };

/* ---- set-up ------------------------------------------------------------------ */

/* Lattice Ns^3 x Nt (both even, >= 2; the checkerboard of P:374 needs even extents), Wilson
 * coupling beta >= 0, 64-bit seed.  Makes a hot start theta ~ U[-pi,pi) from the seed
 * (Philox tag 1, S8(c)-O4) and sets the sweep counter to 0.  UL_EINVAL on bad sizes/beta,
 * UL_ECUDA if no device, UL_ENOMEM if the link array cannot be allocated. */
int ul_create(ul_ctx** h, int Ns, int Nt, double beta, uint64_t seed);

/* Same, on caller-owned DEVICE memory and stream.  dev_links: >= 4*V*4 bytes, 256-byte
 * aligned.  dev_work: workspace for the multilevel accumulators and reduction scratch, may
 * be NULL/0 (then measurement calls cudaMalloc what they need), else it must hold
 * ul_workspace_bytes(...) of the measurement that will be requested (UL_ENOMEM otherwise).
 * cuda_stream: a cudaStream_t (NULL = default stream). */
int ul_create_ext(ul_ctx** h, int Ns, int Nt, double beta, uint64_t seed,
                  void* dev_links, size_t links_bytes,
                  void* dev_work, size_t work_bytes, void* cuda_stream);

/* Bytes of device workspace a measurement needs: accumulators of rows a7-a9 of S8(a)
 * (Ns^3*(Nt/d)*3*r_max complex fp64, times (1 + 12*n_fp) with field points, for each level)
 * plus per-configuration scratch.  d_out = 0 for a single-level measurement. */
size_t ul_workspace_bytes(int Ns, int Nt, int d_in, int d_out, int r_max, int n_fp);

int ul_destroy(ul_ctx* h);

/* mode 0: cold start theta = 0; mode 1: hot start from the seed (same as ul_create). */
int ul_init(ul_ctx* h, int mode);
int ul_set_beta(ul_ctx* h, double beta);

/* Canonical HOST array in / out (see top).  ul_set_links returns UL_EINVAL if any angle is
 * NaN or has |theta| > 3.2 (angles must already be wrapped to [-pi, pi] up to rounding). */
int ul_set_links(ul_ctx* h, const float* host_links);
int ul_get_links(ul_ctx* h, float* host_links);

/* ul_get_links without waiting for the copy (row a1; a serving loop that reads every configuration back): the
 * canonical copy is formed on the context's stream into a library-owned device buffer of its own (4 V floats, allocated on
 * the first call) and copied to host_links on a second stream, so it runs beside whatever is enqueued next, e.g. the
 * ul_set_links of the next configuration (both directions of the host link busy at once).  host_links is caller-owned,
 * should be pinned (with pageable memory the call itself waits), and must not be read or freed before ul_get_links_wait
 * returns UL_OK.  A second call before the wait is allowed: it waits on the stream for the first copy (the buffer is
 * reused), so one wait covers both.  UL_EINVAL on null pointers, UL_ECUDA on a CUDA failure. */
int ul_get_links_async(ul_ctx* h, float* host_links);
int ul_get_links_wait(ul_ctx* h);

/* ul_set_links in two parts, for the same loop: ul_set_links_async copies host_links (caller-owned, pinned, untouched until
 * the commit returns) into a library-owned device buffer of its own (4 V floats, allocated on the first call) on a second
 * stream -- nothing the context's stream is doing is touched, so the upload of the NEXT configuration runs beside the work on
 * the current one; ul_set_links_commit then makes it the configuration: the repack and the validation of ul_set_links on the
 * context's stream, behind the upload (its validation flag sits in mapped host memory: reading it queues no copy behind a
 * ul_get_links_async still in flight).  A second ul_set_links_async before the commit replaces the first.  ul_set_links_commit
 * returns UL_ESTATE without a pending upload, UL_EINVAL for an invalid angle (as ul_set_links; the links are then undefined). */
int ul_set_links_async(ul_ctx* h, const float* host_links);
int ul_set_links_commit(ul_ctx* h);

/* The same arrays as raw binary angles, HOST int32[4][Nt][Ns][Ns][Ns], bit for bit: the exact
 * state for checkpoint / resume (with ul_get_counter / ul_set_counter and the seed). */
int ul_set_links_raw(ul_ctx* h, const int32_t* host_links);
int ul_get_links_raw(ul_ctx* h, int32_t* host_links);

/* 64-bit count of heatbath sweeps issued so far = the Philox counter words 1,2 (S8(c)-O4).
 * State = links + counter + seed: restoring both resumes a run bit for bit. */
int ul_get_counter(ul_ctx* h, uint64_t* sweep_counter);
int ul_set_counter(ul_ctx* h, uint64_t sweep_counter);

/* ---- updates (S8(a) rows a2-a6) -------------------------------------------- */

/* n_hb heatbath sweeps, then n_or overrelaxation sweeps, of the whole lattice.  One sweep =
 * 8 sub-steps: parity outer (even, odd: P:374), direction inner (0..3), in place.  Heatbath
 * draws theta' = alpha + phi, phi ~ exp(beta k cos phi), from the staple sum k e^{i alpha}
 * (DESIGN R2: Best-Fisher rejection; R19: Philox4x32-10 keyed by (seed; site, sweep, block,
 * parity, mu), two attempts per block); overrelaxation sets theta' = 2 alpha - theta.
 * Asynchronous on the stream.  How the sub-steps are launched depends on the lattice and never on
 * the result (bit-identical, tested): one kernel per sub-step with programmatic dependent launch
 * between them; a CUDA graph per recipe on lattices of <= 2^21 sites; one cooperative launch per
 * compound sweep on lattices of <= 256 thread-block tiles (csrc/ul_persist.cuh).  Environment
 * switches, read when the handle is created (for A/B measurements; defaults are the fast paths):
 * UL_NO_PDL=1, UL_NO_ZFLIP=1 (alternating traversal of the time layers), UL_NO_PERSIST=1,
 * UL_PERSIST_VEC=1|2|4, UL_OR_TMA=1 (overrelaxation through the bulk-copy staged gather,
 * csrc/ul_update_tma.cuh: slower), UL_BLOCK_BY=n (x2 row pairs per thread
 * block, the rest of its 128 row pairs along x3; default: an even split), UL_NO_HB_LOCAL=1,
 * UL_GROUP_STREAMS=n. */
int ul_sweep(ul_ctx* h, int n_hb, int n_or);

/* Test hook: one sub-step.  kind 0 = heatbath (draws with the current sweep counter, does
 * not advance it), 1 = overrelaxation, 2 = Metropolis (draws like a heatbath sub-step).
 * slab_d > 0 freezes spatial links (mu != 0) on time layers t % slab_d == 0;
 * 0 = no mask.  Nt % slab_d must be 0. */
int ul_substep(ul_ctx* h, int kind, int parity, int mu, int slab_d);

/* Algorithm of the stochastic ("n_hb") sweeps of ul_sweep and of the sub-updates: 0 = heatbath (default,
 * BASELINE north star), 1 = the paper's Metropolis update ("standard Metropolis algorithm combined with
 * 3 steps of overrelaxation"; DESIGN R21: one hit per link, uniform proposal theta' = theta + delta (2 u1 - 1),
 * accepted iff u2 <= exp(beta k [cos(theta' - alpha) - cos(theta - alpha)]); Philox tag 3).  delta: proposal
 * half-width in radians, 0 < delta <= pi (ignored for alg = 0).  ul_substep takes kind = 2 for a Metropolis
 * sub-step whatever the setting.  UL_EINVAL otherwise. */
int ul_set_update_algorithm(ul_ctx* h, int alg, double delta);

/* Sub-update recipe used inside the multilevel calls: k_sweeps x (n_hb HB + n_or OR) masked
 * sweeps between measurements.  Default 1 HB + 3 OR, k_sweeps = 1 (DESIGN R4, R5). */
int ul_set_subupdate(ul_ctx* h, int n_hb, int n_or, int k_sweeps);

/* ---- multilevel measurement (Alg. 1; S8(a) rows a6-a10, a13) -------- */

/* Single level.  Repeats n_sub times { sub-update with spatial links frozen on layers
 * t % slab_thickness == 0; accumulate T^(d)(x,s,mu,r) (Eq. 22, Eq. 25) for
 * mu = 1..3, r = 1..r_max and, for each field point, T^(d) * sum_{t in slab} O_ch (Eq. 31
 * P:340) }, then forms the slab averages, their product over slabs and the lattice average
 * (Eq. 26, Eq. 34).  n_sub = 0 measures the current configuration once
 * without updating (naive estimator).  field_points: HOST int[n_fp][3] = (a,b,c) in the
 * charge-aligned frame of S8(b): y = x + (floor(r/2)+a) mu + b nu + c rho, nu = 1+(mu mod 3),
 * rho = 1+((mu+1) mod 3); may be NULL with n_fp = 0.
 * UL_EINVAL: Nt % slab_thickness != 0, r_max < 1 or > Ns/2, n_sub < 0, bad field points.
 * UL_ENOMEM: accumulators exceed the caller's workspace / device memory. */
int ul_multilevel(ul_ctx* h, int slab_thickness, int n_sub, int r_max,
                  const int* field_points, int n_fp);

/* Single level by REPLAY (memory formula P:378-384).  The same estimator as
 * ul_multilevel, the same sub-update trajectory, the same outputs (correlators bit for bit, field
 * values to fp64 rounding order) and the same final configuration and sweep counter, but without the
 * per-site TO accumulators, which are 12 n_fp times the T accumulators (972 MB against 1.7 MB in the
 * paper's own example): the estimator is linear in O and the counter-based RNG makes the trajectory
 * repeatable, so pass 1 accumulates only the sums of T, and pass 2 replays the sub-updates from the
 * saved start configuration and adds W(x,s) T_j(x,s) sum_t O_j(x+off,t), W = prod_{s' != s} [T](x,s'),
 * straight into lattice sums.  Costs the sub-update sweeps twice; workspace ul_workspace_bytes_replay
 * (two T-sized arrays).  n_fp = 0 is the same as ul_multilevel.  Errors as ul_multilevel. */
int ul_multilevel_replay(ul_ctx* h, int slab_thickness, int n_sub, int r_max,
                         const int* field_points, int n_fp);
size_t ul_workspace_bytes_replay(int Ns, int Nt, int slab_thickness, int r_max, int n_fp);

/* Two levels by REPLAY (for BJ config 4's field maps): the same estimator, trajectory, outputs and final state as
 * ul_multilevel2 without its TO accumulators.  The weights of the linear-in-O form need the inner averages of the
 * same outer iteration and the outer averages of the whole measurement: pass 1 runs the measurement with the sums
 * of T only; pass 2 restarts from the saved configuration and runs the inner loop of every outer iteration twice
 * (once for [T^(d_in)] and the weights, once to reduce weight x T x O on the fly): about three times the
 * sub-update sweeps.  Workspace: ul_workspace_bytes_replay2 (plus two configuration copies the library allocates). */
int ul_multilevel2_replay(ul_ctx* h, int d_in, int n_in, int d_out, int n_out, int r_max,
                          const int* field_points, int n_fp);
size_t ul_workspace_bytes_replay2(int Ns, int Nt, int d_in, int d_out, int r_max, int n_fp);

/* Two levels (Eq. 27, Eqs. 32-33 P:343-347 with DESIGN R7, Alg. 1 lines 5-18):
 * n_out x { sub-update masked with d_out; n_in x { sub-update masked with d_in; accumulate
 * T^(d_in), TO^(d_in) }; combine the m = d_out/d_in inner slab averages of each outer slab
 * and accumulate }.  Needs d_in | d_out | Nt, n_in >= 1, n_out >= 1. */
int ul_multilevel2(ul_ctx* h, int d_in, int n_in, int d_out, int n_out, int r_max,
                   const int* field_points, int n_fp);

/* Test hooks: open a single-level measurement, add the current configuration to the slab
 * sums (rows a7, a8), close (row a10).  ul_accumulate returns UL_ESTATE if none is open. */
int ul_measure_begin(ul_ctx* h, int slab_thickness, int r_max, const int* field_points, int n_fp);
int ul_accumulate(ul_ctx* h);
int ul_measure_end(ul_ctx* h);
/* The same for two levels (Alg. 1 lines 5, 16, 18; Eqs. 32-33 P:343-347 with DESIGN R7): begin; per outer
 * iteration { ul_accumulate for every inner configuration; ul_combine: inner averages = inner sums / number of
 * configurations accumulated since the last combine, T^(d_out) and TO^(d_out) of every outer slab added to the outer
 * sums, inner sums restarted }; end: outer averages = outer sums / number of combines, slab product, reduction
 * (row a10).  ul_multilevel2 is this sequence with its own sub-updates in between.  UL_ESTATE: no two-level
 * measurement open, nothing accumulated since the last combine, a different number of configurations than in
 * the previous outer iteration, configurations pending at end; ul_measure_end refuses a two-level measurement. */
int ul_measure2_begin(ul_ctx* h, int d_in, int d_out, int r_max, const int* field_points, int n_fp);
int ul_combine(ul_ctx* h);
int ul_measure2_end(ul_ctx* h);

/* Slab-group-major order of the sub-update loop ("hold their spatial links constant [and] isolate the dynamics
 * of the sublattice from the rest of the lattice").  The slabs are dynamically independent during the n_sub loop of
 * ul_multilevel, so the loop may run slab group by slab group: all n_sub masked sub-updates, tables and accumulation
 * passes of `n_slabs` consecutive slabs, then the next group -- the group's links and tables stay in L2 instead of
 * streaming the whole lattice from HBM for every sub-step.  Counter-based RNG and per-entry accumulation make the
 * links, the sweep counter, the slab sums, C(r) and G bit-identical to the sub-update-major order (tested); only the
 * vacuum sums are added in a different order (1e-16 relative).  n_slabs = 0: off; -1 (default): automatic (rounds of
 * ~64 MB of links in flight, split over the group streams below, on lattices whose links exceed 96 MB: 12.6 % faster on
 * 64^4); > 0: that many slabs per group.  UL_ESTATE: a measurement is open.
 * ul_substep_slabs is the test hook underneath: ul_substep restricted to the slabs s_begin <= s < s_end of
 * thickness slab_d >= 1 (UL_EINVAL on a bad range). */
int ul_set_slab_group(ul_ctx* h, int n_slabs);
/* Slab groups per round of the slab-group-major loop: n_streams groups run side by side, each on its own stream (own
 * straggler queue and sweep-counter copy), one compound sub-update of a round captured once as a CUDA graph and replayed.
 * 1 = one group after the other; default 4.  Bit-identical results.  UL_EINVAL outside 1..8; UL_ESTATE: a measurement is
 * open. */
int ul_set_slab_group_streams(ul_ctx* h, int n_streams);
int ul_substep_slabs(ul_ctx* h, int kind, int parity, int mu, int slab_d, int s_begin, int s_end);

/* Analytic multihit inside the two-link operators: with on = 1 the sums of
 * T^(d)(x,s,r mu) for r >= 2 are built from multihit temporal links Ubar_0 = (I1(beta k)/I0(beta k)) e^{i alpha}
 * (k e^{i alpha} the staple sum) instead of U_0: the same expectation value, a smaller variance.  r = 1 keeps the
 * plain links (the two lines share plaquettes there), and so do all TO sums (a plaquette next to a line would be
 * biased).  Applies to ul_multilevel, ul_multilevel2, ul_multilevel_replay and the ul_accumulate hook; needs
 * 16 * depth * (Nt/d) * Ns^3 more workspace bytes than ul_workspace_bytes (depth = accumulation batch depth).
 * UL_EINVAL: on not 0 or 1; UL_ESTATE: a measurement is open. */
int ul_set_multihit(ul_ctx* h, int on);

/* Accumulation batch depth (rows a7, a8).  The library tabulates up to `depth` configurations
 * (exp(i sum_t theta_0) per slab and site, and the plaquette sums) and adds them to the slab sums
 * in ONE read-modify-write pass, in sub-update order: the same sequence of fp64 additions as
 * `depth` single passes, so results do not depend on it (tested bit for bit).  depth = 0 restores
 * the default (8, less when the tables would outgrow the accumulators); values above the default
 * are clamped.  Takes effect at the next measurement.  UL_EINVAL: depth < 0. */
int ul_set_accum_batch(ul_ctx* h, int depth);

/* Mean of cos theta_P (Eq. 6) over all 6V plaquettes, over the 3V time-like and the
 * 3V space-like ones: HOST double[3].  Synchronises. */
int ul_plaquette(ul_ctx* h, double* mean_cos);
/* The same numbers (bit for bit: same kernels, same order of additions) for callers that must not allocate -- code under
 * CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Input: the handle's current links; output:
 * DEVICE double[3] (caller-owned), written asynchronously on the handle's stream (no synchronisation, no host copy).
 * Calls no cudaMalloc / cudaFree / allocating routine: the block partials live in a fixed file-scope device array of
 * 2 * 592 + 4 doubles (9.5 KB, held by every GPU that loads the library until exit).  Limit: ceil(Ns^2 / 256) <= 592,
 * i.e. Ns <= 389 (any Nt); beyond it UL_EINVAL with a message that says so.  The first call on a device looks the array's
 * address up (cudaGetSymbolAddress: make one call outside capture first).  EVERY call on a device, of any handle, shares
 * that array, which keeps the last call's contents (each call overwrites all it reads, nothing needs clearing): calls that
 * can overlap on the GPU (different streams) race -- order them.  UL_EINVAL: null pointers, device index beyond 63. */
int ul_plaquette_noalloc(ul_ctx* h, double* dev_mean_cos);

/* Polyakov-loop average <P> = (1/Ns^3) sum_x prod_t U_0(x,t) (Eqs. 15-16): HOST double[2] = (Re, Im).
 * multihit = 1: analytic multihit, every temporal link replaced by its mean over its local weight with the
 * other links fixed, U_0 -> (I1(beta k)/I0(beta k)) e^{i alpha}, k e^{i alpha} the staple sum (
 * SURVEY S8(f) rank 1); same expectation value, smaller variance.  fp64 throughout.  Synchronises.
 * UL_EINVAL: multihit not 0 or 1, null pointer. */
int ul_polyakov(ul_ctx* h, int multihit, double* mean_P);

/* ---- slab sharding over GPUs -------------------------
 * While the boundary layers are frozen the slabs are dynamically independent, so a lattice can be cut
 * in t into shards of whole slabs, one ul_ctx per GPU, with NO communication inside the sub-update loop:
 * a shard is a lattice of Nt_loc + d time layers whose last slab is a ghost (its first layer holds a copy
 * of the next shard's frozen spatial links; nothing a shard owns depends on the rest of the ghost slab).
 * ul_set_site_offset makes the Philox counters those of the global lattice (offset = t0 * Ns^3 added to
 * the local site index; it may be negative, down to -V, when ghost layers sit below the shard's first own layer;
 * offset + local volume <= 2^29), so a sharded run reproduces the unsharded one bit
 * for bit.  ul_slab_partial_product writes prod_{s_begin <= s < s_end} [T](x,s) of the last measurement
 * to a DEVICE buffer double[3][r_max][Ns^3][2] (caller-owned, e.g. a torch tensor): the one array the
 * shards exchange (all-gather) before the slab product of row a10.  paper_1309_3859_b200/sharded.py holds
 * the partition arithmetic and the exchange over torch.distributed. */
int ul_set_site_offset(ul_ctx* h, int64_t offset);
int ul_slab_partial_product(ul_ctx* h, int s_begin, int s_end, void* dev_out);
/* The last step of row a10 across shards (Eq. 24, Eq. 26): dev_parts[k], k = 0..n_parts-1 in rank
 * order, are DEVICE buffers double[3][r_max][Ns^3][2] on this context's GPU (the own ul_slab_partial_product and the
 * copies received from the other ranks; caller-owned); the kernel multiplies them in that order, site by site, and
 * sums over the lattice and the three directions with the library's fixed two-stage tree (bitwise reproducible):
 * corr[r_max][2] (HOST) = C(r) of the whole lattice, which ul_read_correlators returns from then on.  r_max is that of
 * the last measurement.  Synchronises.  UL_ESTATE before any measurement; UL_EINVAL: null pointers, n_parts
 * outside 1..64. */
int ul_combine_partial_products(ul_ctx* h, const void* const* dev_parts, int n_parts, double* corr);

/* ---- t-sharded FULL sweeps with peer-memory halo writes ---------------------------
 * A shard of a lattice cut in t holds ghost_layers (even, >= 2) ghost time layers below and above its own layers.  With
 * the neighbours' link arrays set here -- DEVICE pointers to the internal-layout arrays of the shards below (t - 1 side)
 * and above, of the same local shape: memory of the same device, or of another device of this process (peer access is
 * enabled here; NVLink on B200) -- every unmasked sub-step kernel updates the own layers only and stores the first /
 * last ghost_layers own layers it has just computed ALSO into the neighbours' ghost layers: one fused kernel per
 * sub-step, no exchange step.  Ordering between neighbours is stream-ordered, without host synchronisation and without
 * spinning kernels: before a sub-step the stream waits (cuStreamWaitValue32) until both neighbours have reported the
 * previous sub-step complete; after it, it reports to both (cuStreamWriteValue32 into their flag words).  ul_halo_flags
 * returns (and zeroes) this context's two flag words; ul_set_halo_peer_flags takes the neighbours' (the pointers their
 * ul_halo_flags returned) -- without it no waits or reports are issued and the caller orders the shards (e.g. one
 * stream).  All shards must issue the same sequence of sub-steps.  (NULL, NULL) switches the mode off.
 * UL_EINVAL: one neighbour missing, odd or too many ghost layers, pointers that are not device memory; UL_ECUDA: no peer
 * access between the devices; UL_ESTATE: a measurement is open / ul_halo_flags not called before ul_set_halo_peer_flags. */
int ul_set_halo_peers(ul_ctx* h, void* dn_links, void* up_links, int ghost_layers);
int ul_halo_flags(ul_ctx* h, void** dev_flags);
int ul_set_halo_peer_flags(ul_ctx* h, void* dn_flags, void* up_flags);
/* The same between processes (one process per GPU, the shards' processes exchange the 64-byte handles through
 * torch.distributed): ul_ipc_export writes the CUDA IPC handles (cudaIpcMemHandle_t, 64 bytes each) of the allocations
 * that hold this context's link array and its flag words (ul_halo_flags first) and the byte offsets of the two inside
 * them; ul_ipc_open maps a neighbour's allocation into this process (once per allocation; closed by ul_destroy) and
 * returns the device pointer to pass to ul_set_halo_peers / ul_set_halo_peer_flags.  The exporting memory must come
 * from cudaMalloc (ul_create, or a PyTorch tensor of the default caching allocator).  UL_ECUDA if IPC is refused. */
int ul_ipc_export(ul_ctx* h, void* out_links_handle, uint64_t* links_offset, void* out_flags_handle, uint64_t* flags_offset);
int ul_ipc_open(ul_ctx* h, const void* handle, uint64_t offset, void** dev_ptr);

/* Results of the last measurement, HOST buffers (any may be NULL):
 * corr[r_max][2]           C(r) = (1/3Ns^3) sum_x sum_mu prod_s [T](x,s,mu,r)       (re, im)
 * field[r_max][n_fp][12][2] G(r,fp,ch) of Eq. 34; ch = 2*comp + kind, comp 0..5 = plaquette
 *                          orientations (0,mu) (0,nu) (0,rho) (nu,rho) (rho,mu) (mu,nu),
 *                          kind 0 = 1 - cos theta_P, 1 = sin theta_P (Eqs. 28-29
 *                          without the beta factors)
 * vacuum[12]               <O_ch> over all sites, times and the three frames: the mean over the measured
 *                          configurations when field points were requested; with n_fp = 0 (nothing to
 *                          subtract from, Eq. 30) the plaquettes are not evaluated per sub-update and
 *                          the values are those of the final configuration of the measurement.
 * UL_ESTATE before any measurement.  Synchronises. */
int ul_read_correlators(ul_ctx* h, double* corr, double* field, double* vacuum);

/* Slab averages [T] of the last measurement (outer level for two levels), HOST
 * double[3][r_max][n_slab][Ns^3][2], xs = x1 + Ns*(x2 + Ns*x3).  Test hook for parity P2. */
int ul_read_slab_averages(ul_ctx* h, double* out);

/* Number of kernels this handle has launched since creation (bench.py's gpu_launches). */
int ul_get_launch_count(ul_ctx* h, uint64_t* n);

/* Philox4x32-10 known-answer hook: runs the DEVICE generator on n (ctr[4], key[2]) tuples.
 * HOST pointers: ctr uint32[n][4], key uint32[n][2], out uint32[n][4]. */
int ul_philox_selftest(const uint32_t* ctr, const uint32_t* key, uint32_t* out, int n);

/* Blocks until everything enqueued on the handle's stream has finished. */
int ul_sync(ul_ctx* h);

const char* ul_last_error(ul_ctx* h);

#ifdef __cplusplus
}
#endif
#endif
