/* mc.h — C ABI of the B200-native coupled photon–electron Monte Carlo dose engine.
 *
 * The calls follow the paper's statement of the problem (arxiv 1503.01722, "oclMC"):
 *   - a voxelised phantom, "each voxel was assigned to a density value and a material type"
 *     (§2.1)                                            -> mc_create
 *   - "physics data needed by oclMC based on a user-defined material composition", cut-offs and
 *     maximum step sizes are user defined    -> mc_build_tables / mc_set_photon_tables
 *   - a point source with an energy or spectrum, a field at the surface, an SSD;
 *     result "in a unit of MeV/g per source particle" with its uncertainty sigma_D
 *                                                                     -> mc_run
 * Transport: photons by Woodcock tracking with Compton / pair / photoelectric events,
 * electrons and positrons by a Class II condensed-history scheme with
 * d = min[d_vox, d_maxs, d_maxe, d_event], secondaries on per-type stacks
 * (PAPER.md:60, :72), dose by atomic adds.  Readings of everything the paper leaves
 * open are listed in DESIGN.md (R1..R28, with R8b and R13b).
 *
 * Conventions
 *   - Every call returns an mc_status and never throws or aborts; mc_last_error() gives a message.
 *   - Plain pointers and sizes only.  Unless stated otherwise an input pointer is HOST memory that is
 *     copied during the call (the caller keeps ownership); an output pointer may be HOST or DEVICE
 *     memory (resolved through unified addressing) and is written before the call returns.
 *   - The context owns all device memory it allocates.  One context = one phantom on the current
 *     CUDA device; calls on one context must not overlap.  Work is issued on the context's stream
 *     (default: the legacy default stream; see mc_set_stream) and the call synchronises that stream
 *     before returning.
 *   - Volume layout: x fastest, i = ix + nx*(iy + ny*iz).  Units: MeV, cm, g/cm^3.
 *   - There is no CPU fallback: without a CUDA device every compute call returns MC_ERR_CUDA.
 */
#ifndef MC_B200_H
#define MC_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mc_ctx mc_ctx; /* opaque, owned by the library */

typedef enum {
    MC_OK = 0,
    MC_ERR_INVALID_ARG = 1,
    MC_ERR_STATE = 2,          /* e.g. mc_run before tables exist                        */
    MC_ERR_ENERGY_RANGE = 3,   /* beam energy above the table grid (e_max_MeV)           */
    MC_ERR_QUEUE_OVERFLOW = 4, /* a particle queue overflowed: results invalid, none returned */
    MC_ERR_OOM = 5,
    MC_ERR_CUDA = 6
} mc_status;

/* One material by elemental composition.  Z, A, w: n_elem entries; w = mass fractions
 * (normalised by the library).  I_eV = mean excitation energy; rho_nominal (g/cm^3) enters only the
 * density-effect correction (R22). */
typedef struct {
    int32_t n_elem;
    const int32_t *Z;
    const float *A;
    const float *w;
    float I_eV;
    float rho_nominal;
} mc_material;

/* flags */
#define MC_FLAG_NO_HARD_EVENTS 1u     /* no Moller / bremsstrahlung events (d_event = inf)        */
#define MC_FLAG_NO_MS 2u              /* no multiple-scattering deflection                        */
#define MC_FLAG_LOCAL_SECONDARIES 4u  /* secondaries deposit their energy where they are born     */
#define MC_FLAG_MS_GS 8u              /* multiple-scattering angle from the Goudsmit-Saunderson distribution of the
                                         screened-Rutherford law ("the method developed by Kawrakow";
                                         DESIGN.md R27) instead of the Gaussian model (R7)                        */

#define MC_FLAG_MULTI_VOXEL 16u       /* electron steps are not limited by the voxel: a step of length
                                         min[d_maxs, d_maxe, d_range, d_event] crosses voxel faces (the stepping of
                                         gDPM the paper compares with; R28) instead of
                                         d = min[d_vox, ...]                                        */

/* Cut-offs and step limits (PAPER.md:39 "user defined maximum step size", :86 cut-off energies).
 * e_cut_MeV: electron absorption energy = Moller delta-ray threshold; g_cut_MeV: photon absorption
 * energy = bremsstrahlung production threshold (R1).  e_max_MeV: top of the energy grid.
 * n_grid: nodes of the uniform ln E grid (8..1024).  d_maxs_cm: geometric step limit; f_maxe:
 * maximum fractional CSDA energy loss per step (R2). */
typedef struct {
    float e_cut_MeV, g_cut_MeV, e_max_MeV;
    int32_t n_grid;
    float d_maxs_cm, f_maxe;
    uint32_t flags;
} mc_params;

#define MC_PHOTON 0
#define MC_ELECTRON (-1)
#define MC_POSITRON 1
#define MC_SHAPE_PENCIL 0     /* all histories start at entry_cm along axis                              */
#define MC_SHAPE_POINT_RECT 1 /* point source at ssd_cm behind entry_cm; (x, y) uniform over field_cm in
                                 the surface plane z = entry_cm[2]; axis must be +z (R13)       */

/* Beam.  Spectrum: n_nodes == 1 -> monoenergetic E_nodes_MeV[0]; otherwise a
 * piecewise-linear pdf through (E_nodes_MeV[j], pdf_nodes[j]), nodes ascending. */
typedef struct {
    int32_t particle;
    int32_t shape;
    float entry_cm[3];
    float axis[3];
    float ssd_cm;
    float field_cm[2];
    int32_t n_nodes;
    const float *E_nodes_MeV;
    const float *pdf_nodes;
} mc_beam;

/* Counters of the last mc_run / mc_run_range on this context. */
typedef struct {
    uint64_t n_histories;
    uint64_t n_electron_steps;   /* condensed-history steps (electrons + positrons)            */
    uint64_t n_photon_flights;   /* Woodcock flights                                           */
    uint64_t n_fictitious;       /* flights ending in a fictitious interaction                 */
    uint64_t n_compton, n_pair, n_photoelectric;
    uint64_t n_moller, n_brems;
    uint64_t n_secondary_electrons, n_secondary_photons; /* queued (not counting local deposits) */
    uint64_t n_dose_atomics;     /* red.global.add.f32 issued                                  */
    uint64_t n_kernel_launches;  /* transport + finalize kernels launched                      */
    double e_source_MeV, e_deposited_MeV, e_escaped_MeV; /* energy ledger                      */
    double transport_ms;         /* CUDA-event time of the transport launches                  */
    double electron_kernel_ms, photon_kernel_ms; /* split of transport_ms by kernel            */
    uint64_t n_host_syncs;       /* counter read-backs (stream synchronisations) inside the transport loop */
} mc_stats;

/* mc_create — copy the phantom to the device.
 * material_idx, density_gcc: nx*ny*nz entries (host), density > 0.  1 <= dims <= 1024 per axis (a track carries
 * its voxel indices in one 32-bit word), voxel_cm > 0.
 * origin_cm: coordinates of the low corner of voxel (0,0,0).  *out receives the context. */
mc_status mc_create(const uint8_t *material_idx, const float *density_gcc, const int32_t dims[3],
                    const float voxel_cm[3], const float origin_cm[3], mc_ctx **out);
void mc_destroy(mc_ctx *ctx);

/* mc_build_tables — closed-form physics tables per material on a uniform ln E grid, the photon
 * Woodcock majorant from the phantom.  Re-callable.
 * n_mats: 1..16 (tables and track pools share the 227 KB of shared memory: 3 materials x 256 nodes run on the largest CTAs,
 * 16 materials need n_grid <= 128).  Errors: a voxel's material index >= n_mats, bad cut-offs / grid -> MC_ERR_INVALID_ARG. */
mc_status mc_build_tables(mc_ctx *ctx, const mc_material *mats, int32_t n_mats, const mc_params *params);

/* Table access, fp32 as used on the device.  which: 0 mu_tot 1 mu_C 2 mu_pp (cm^2/g) 3 R (g/cm^2)
 * 4 L (MeV cm^2/g) 5 Sigma_hard 6 Sigma_Moller 7 Sigma_max 8 K1 (cm^2/g); material = -1, which = 9:
 * photon majorant mu_maj (1/cm).  out: n_grid floats (host). */
mc_status mc_export_table(const mc_ctx *ctx, int32_t material, int32_t which, float *out);
/* which = 10: ln of the effective screening parameter of the Goudsmit-Saunderson model (R27).
 * mc_export_gs_table — the material-independent Goudsmit-Saunderson sampling table (R27): dims = {NT, NA, NQ};
 * t_nodes[NT] (may be NULL) the scattering-power nodes; y[NT*NA*NQ] (may be NULL) ln of the quantiles of
 * 1 - cos(theta).  Host pointers; needs no context and no device (the table is built on the host). */
mc_status mc_export_gs_table(int32_t dims[3], float *t_nodes, float *y);
/* grid[0] = ln E_0, grid[1] = delta ln E, grid[2] = n_grid, grid[3] = node index of e_cut. */
mc_status mc_export_grid(const mc_ctx *ctx, double grid[4]);
/* Replace the PHOTON tables by user-supplied data ("physics data ... stored in a database",
 * PAPER.md:31): mu_maj[n_grid] (1/cm) and mu_tot / mu_C / mu_pp [n_mats][n_grid] (cm^2/g) on the grid
 * ln E_j = lnE0 + j/inv_dln.  Requires a previous mc_build_tables with the same n_mats and n_grid. */
mc_status mc_set_photon_tables(mc_ctx *ctx, float lnE0, float inv_dln, const float *mu_maj,
                               const float *mu_tot, const float *mu_C, const float *mu_pp);

/* mc_run — simulate histories 0..n_histories-1 (n_histories < 2^32) of the beam with Philox4x32-10
 * streams keyed by (seed, history index), scoring into n_batches (>= 2, <= n_histories) per-batch
 * fp32 grids (batch of history h = floor(h*n_batches/n_histories)).
 * dose_out, sigma_out: nvox floats each (host or device): mean dose and standard error of the batch
 * means, MeV/g per history (R17, R18).  Results are deterministic per history; grid sums
 * are reproducible only to fp32 summation order. */
mc_status mc_run(mc_ctx *ctx, const mc_beam *beam, uint64_t n_histories, uint64_t seed, int32_t n_batches,
                 float *dose_out, float *sigma_out);

/* One source particle of a particle list (a phase-space record; PAPER.md:84 leaves the source interface open:
 * "phase-space file" or a "user ... function").  particle: 0 photon, -1 electron, +1 positron; position in cm in
 * phantom coordinates; (u, v, w) a unit vector; E kinetic energy in MeV (<= e_max_MeV). */
typedef struct {
    float x, y, z, u, v, w, E;
    int32_t particle;
} mc_particle;

/* mc_run_particles — as mc_run, but the source is a list: history h is particles[h], transported with track id (0,0)
 * from Philox block 0 (R13b).  A particle outside the phantom counts as escaped (no re-entry, R3).
 * particles: n records, HOST or DEVICE memory (a host list is validated on the host and staged; a device list is
 * validated by one kernel pass and read in place).  Errors: an energy outside (0, e_max_MeV] -> MC_ERR_ENERGY_RANGE, a
 * direction that is not a unit vector or an unknown particle type -> MC_ERR_INVALID_ARG; otherwise as mc_run. */
mc_status mc_run_particles(mc_ctx *ctx, const mc_particle *particles, uint64_t n, uint64_t seed, int32_t n_batches,
                           float *dose_out, float *sigma_out);

/* mc_run_source — as mc_run_particles, but the records come from a user function ("a user can either load source
 * particles from a phase-space file or write a CPU/GPU function"): the library calls
 *     fn(user, h_begin, n, out, cuda_stream)
 * once per wave of histories [h_begin, h_begin + n) (n <= option "wave_size", waves in ascending order); the function
 * writes records h_begin .. h_begin + n - 1 to out — DEVICE memory owned by the library, valid during the call — and
 * returns 0 (anything else aborts the run with MC_ERR_INVALID_ARG).  The writes must be ordered before the library's
 * use of the records, which happens on cuda_stream (a cudaStream_t: the context's stream, see mc_set_stream).  Three
 * ways satisfy that: (1) work enqueued on cuda_stream itself — a kernel of the function's own or cudaMemcpyAsync(...,
 * cuda_stream) — needs no synchronisation; (2) a plain cudaMemcpy / work on the LEGACY default stream: the library makes
 * cuda_stream wait for everything the function left on the legacy stream (this matters when mc_set_stream installed a
 * non-blocking stream: a copy from pageable host memory may return before its DMA has landed); (3) anything else (another
 * stream, a per-thread default stream) must be complete on the device before the function returns.  A host buffer
 * handed to an asynchronous copy must stay valid until that copy is done.  Records are validated on the device as for a
 * device-resident list. */
typedef int (*mc_source_fn)(void *user, uint64_t h_begin, uint64_t n, mc_particle *out, void *cuda_stream);
mc_status mc_run_source(mc_ctx *ctx, mc_source_fn fn, void *user, uint64_t n, uint64_t seed, int32_t n_batches,
                        float *dose_out, float *sigma_out);

/* mc_run_range — the shard of mc_run one GPU of several computes: histories [h_begin, h_end) of a
 * job of n_histories.  edep_out: n_batches*nvox floats (host or device), energy deposited per batch
 * grid in MeV (sum these over shards, then call mc_finalize). */
mc_status mc_run_range(mc_ctx *ctx, const mc_beam *beam, uint64_t n_histories, uint64_t h_begin,
                       uint64_t h_end, uint64_t seed, int32_t n_batches, float *edep_out);
/* mc_finalize — batch statistics kernel: edep [n_batches][nvox] (host or device) -> dose, sigma. */
mc_status mc_finalize(mc_ctx *ctx, const float *edep, uint64_t n_histories, int32_t n_batches,
                      float *dose_out, float *sigma_out);

/* Fused exchange + statistics for the sharded job: instead of summing the ranks' grids with an
 * all-reduce and then calling mc_finalize, every rank (or one) reads all grids in place, over NVLink for a peer's.
 *   mc_edep_buffer     the context's own [n_batches][nvox] grid buffer (device memory, plain cudaMalloc: exportable);
 *                      pass it as edep_out of mc_run_range to leave the shard's grids there without a copy.
 *   mc_ipc_get_handle  CUDA IPC handle (64 bytes) of a device buffer, to be sent to the other ranks by any means.
 *   mc_ipc_open_handle maps another process's buffer into this one (peer access is enabled as needed);
 *   mc_ipc_close_handle unmaps it.
 *   mc_finalize_multi  dose and sigma of the SUM of n_grids (1..16) grids: edep_grids[r] = device-accessible pointer to
 *                      n_batches*nvox floats (own, or opened with mc_ipc_open_handle); edep_grids itself is a HOST array.
 * The caller orders the calls across ranks (all shards finished before any rank finalizes; nobody reuses its buffer
 * before all have finalized), e.g. with torch.distributed.barrier(). */
mc_status mc_edep_buffer(mc_ctx *ctx, int32_t n_batches, float **out);
mc_status mc_finalize_multi(mc_ctx *ctx, const float *const *edep_grids, int32_t n_grids, uint64_t n_histories,
                            int32_t n_batches, float *dose_out, float *sigma_out);
/* mc_finalize_multi_range — the same for voxels [v_begin, v_end) only: dose_out / sigma_out receive v_end - v_begin
 * floats.  With one slice per rank (sharding.voxel_slice) every grid value is read over NVLink exactly once — the
 * reduce-scatter shape of the exchange — and the dose / sigma slices (2 x nvox x 4 bytes in total) are all-gathered. */
mc_status mc_finalize_multi_range(mc_ctx *ctx, const float *const *edep_grids, int32_t n_grids, uint64_t n_histories,
                                  int32_t n_batches, int64_t v_begin, int64_t v_end, float *dose_out, float *sigma_out);
mc_status mc_ipc_get_handle(const void *dev_ptr, uint8_t handle[64]);
mc_status mc_ipc_open_handle(const uint8_t handle[64], void **dev_ptr);
mc_status mc_ipc_close_handle(void *dev_ptr);

/* mc_run_atten — attenuation-only mode (R20): photon primaries only; per history the
 * linear voxel index of the first real interaction (-1 = left the phantom or never interacted) and its
 * channel (0 Compton, 1 pair, 2 photoelectric, 255 none).  fp32 arithmetic contract: bit-exact
 * against any other implementation of the contract given the same tables.
 * voxel_out: n int32; channel_out: n uint8 (host or device; channel_out may be NULL). */
mc_status mc_run_atten(mc_ctx *ctx, const mc_beam *beam, uint64_t n, uint64_t seed, int32_t *voxel_out,
                       uint8_t *channel_out);

/* mc_edep_total_static — the energy-ledger total (what mc_stats.e_deposited_MeV reports: the fp64 sum of the per-batch
 * energy grids that dose is scored into with atomic adds) for callers that are not allowed to allocate GPU
 * memory.  Examples: a host application whose tensor framework has already claimed almost all device memory for its own
 * caching allocator, so a raw cudaMalloc fails; a thread that runs while another thread of the process records a CUDA
 * graph in the global capture mode, during which cudaMalloc / cudaFree are illegal and break the recording; a loop that
 * checks the ledger between beam segments and cannot take the device-wide stall cudaMalloc / cudaFree cause.  Every other
 * compute call of this library builds device state behind a context; this call needs no context and makes no cudaMalloc,
 * cudaFree, memory-pool or other allocating call — the caller passes the input and the output, and the partial sums live
 * in a fixed 512.25 KiB array inside the library's device image (held on every GPU that loads the library until the
 * process exits).
 *   edep_dev     n floats in DEVICE memory (e.g. the buffer of mc_edep_buffer after mc_run_range: n = n_batches * nvox)
 *   n            1 .. mc_edep_total_static_max() = 2^28 floats; anything larger returns MC_ERR_INVALID_ARG (nothing is
 *                summed partially) — split the input and add the totals
 *   total_out    one double, HOST or DEVICE memory, written before the call returns
 *   cuda_stream  a cudaStream_t (0 = default stream); the call enqueues a 16-byte clear, one kernel and an 8-byte copy
 *                there and synchronises that stream
 *   err, err_len optional caller-owned buffer that receives a message when the status is not MC_OK (may be NULL / 0)
 * The sum is taken in a fixed order (one partial per 4096 consecutive floats, partials added in index order), so the
 * same input gives the same bits on every call and every grid size; it differs from e_deposited_MeV only by fp64
 * rounding order.
 * First call on a device: it looks up the array's device address (once per device, with that device current), which is
 * also what loads the library's kernels onto that device — make this first call before starting any stream capture.
 * Shared state: all calls on a device use the one array, which keeps the previous call's contents; the call clears the
 * only word that must start at zero itself.  Two calls on the same device that overlap on the GPU (from two host threads
 * or streams) race on it and return wrong totals — serialise them.
 * Errors: null pointers, n = 0, n above the limit, edep_dev not device memory -> MC_ERR_INVALID_ARG; no device or a CUDA
 * failure -> MC_ERR_CUDA.  Nothing is written to total_out on error. */
mc_status mc_edep_total_static(const float *edep_dev, uint64_t n, double *total_out, void *cuda_stream, char *err,
                               int32_t err_len);
uint64_t mc_edep_total_static_max(void);

/* ---- Diagnostics: test and measurement hooks, not part of the hot path -------------------------------------------
 * (mc_philox_selftest, mc_u01_selftest, mc_bench_red, mc_bench_issue: used by tests/ and bench.py only.) */
/* Philox4x32-10 on the device: n blocks, ctr[4n], key[2n] -> out[4n] (host pointers). */
mc_status mc_philox_selftest(const uint32_t *ctr, const uint32_t *key, int32_t n, uint32_t *out);

/* mc_u01_selftest — the device's uniform-from-word function (two instructions, no integer-to-float conversion) against
 * its definition ((w >> 9) + 0.5) * 2^-23 (R15) for all 2^23 values: *n_mismatch (host) = words that differ. */
mc_status mc_u01_selftest(uint64_t *n_mismatch);

/* mc_bench_red — measures the scoring roofline: `blocks` x 256 threads each
 * issue per_thread red.global.add.f32 into a window of n_cells floats.  mode 0: pseudo-random cell per
 * thread (no intra-warp collisions on average); mode 1: one cell per warp (full intra-warp collision).
 * *ms_out (host) = CUDA-event time of the launch. */
mc_status mc_bench_red(mc_ctx *ctx, uint32_t n_cells, int32_t per_thread, int32_t mode, int32_t blocks,
                       double *ms_out);

/* mc_bench_issue — measures the transport roofline's denominator: 2 x 1024-thread CTAs per SM each run iters x 64
 * independent FFMAs per thread; *thread_instr_per_s (host) = FFMA thread-instructions per second achieved. */
mc_status mc_bench_issue(mc_ctx *ctx, int32_t iters, double *thread_instr_per_s);

/* ---- end of diagnostics ------------------------------------------------------------------------------------------- */

/* mc_trim — the particle queues (gigabytes) come from a memory pool the library keeps per device so that the next
 * context of the process reuses them; mc_destroy returns them to that pool, not to the driver, and memory in a private
 * pool is invisible to every other allocator of the process.  mc_trim hands the unused part of the current device's pool
 * back to the driver, keeping at most keep_bytes (0 = everything unused).  It synchronises the device.  Queues of live
 * contexts are not touched. */
mc_status mc_trim(uint64_t keep_bytes);

mc_status mc_get_stats(const mc_ctx *ctx, mc_stats *out);
/* cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); 0 = default stream. */
mc_status mc_set_stream(mc_ctx *ctx, void *cuda_stream);
/* Tuning knobs ("the number of workitems M ... manually adjusted").  Scheduling only: per-history results
 * do not depend on them (R14).
 *   "wave_size"     histories admitted per launch at most (default 2^24)
 *   "queue_factor"  capacity of each particle queue in waves (default 4)
 *   "adaptive"      1 (default): the number of new primaries a launch admits is limited by the room left in the output
 *                   queues at the measured secondaries-per-primary ratio; 0: always a full wave
 *   "hard_lanes"    tracks of a warp's pool that must wait for the hard-event / Compton block before the warp runs it
 *                   (default 32 = a full warp; the block also runs when it has more tracks than the step block)
 *   "refill_lanes"  empty slots of a warp's pool that trigger a refill from the queue / the source (default 32)
 *   "plan_ahead"    1 (default): once the secondaries-per-primary ratios of the beam are known (a probe launch, or the
 *                   previous run with the same kind of beam) the launches of a run are enqueued ahead — every kernel
 *                   reads the size of its input queue on the device and leaves it empty — and the host reads the
 *                   counters back only once per round of the final cascade; 0: one read-back per launch
 *   "electron_threads" cap on the electron kernel's CTA size: 256, 512, 768 or 1024 (0 = default: the largest of 1024 / 768 / 512 / 256
 *                   threads whose tables and track pools fit in shared memory)
 *   "blocks_per_sm" cap on the CTAs per SM (0 = as many as fit; the transport kernels use one)
 *   "aggregate"     1: lanes of a warp that score into the same cell at the same moment combine into one
 *                   red.global.add.f32; 0: one per lane; -1 (default): 1 for beams entering through fewer than 16
 *                   voxel columns, else 0
 * Readings of the method (R8, R8b; the oracle has the same two switches, used by A/B tests):
 *   "hinge_overrun_pct"  the second leg of a voxel-limited step may run on to the face by this percentage of its
 *                   planned length (default 25; 0 = the plain rule)
 *   "ms_carry"      1 (default): the multiple-scattering angle of a step is sampled for the planned path plus the path
 *                   travelled but not yet sampled for (steps a voxel face cut short or lengthened); 0: planned path only */
mc_status mc_set_option(mc_ctx *ctx, const char *name, int64_t value);
const char *mc_last_error(const mc_ctx *ctx);
const char *mc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MC_B200_H */
