/* rt.h — C ABI of the B200 forward Monte Carlo shortwave photon tracer.
 *
 * Operation: PAPER.md §2.3 "The ray tracer" as read in DESIGN.md §2-§3:
 * photons start at the domain top along the sun beam, fly by single-level
 * null-collision tracking on a coarse acceleration grid whose cell value is the highest
 * extinction coefficient inside the cell, fetch local optical properties from the
 * fine grid, scatter by Rayleigh or Henyey-Greenstein with the cloud/gas split
 * k_ext,cloud/k_ext, reflect at a Lambertian surface with local albedo and
 * are tallied as surface flux (direct = never scattered), domain-top upward flux
 * and 3D absorbed power.  Absorption is analog by default (BASELINE.json north_star):
 * each photon carries RT_W0 = 2^32 integer quanta and ends in exactly one bin.  Options, all off
 * after rt_create_grid: merged acceleration cells (rt_set_merge), the paper's weights + Russian
 * roulette (rt_set_mode), its top-of-domain source (rt_set_source), the direct part of the heating
 * (rt_set_heating_split), many spectral points in one launch (rt_set_slots, rt_trace_batch).
 *
 * Every step runs in CUDA kernels for sm_100a; there is no CPU fallback.  All functions
 * return 0 (RT_OK) or a negative RT_E* code; no exception crosses this boundary;
 * rt_last_error() gives the text of the last failure on that context.
 *
 * Layouts: 3D fields are [z][y][x] with x fastest, z = 0 at the surface; 2D fields are
 * [y][x].  x = east, y = north.  Lateral boundaries are periodic.
 */
#ifndef PAPER_2208_05247_RT_H
#define PAPER_2208_05247_RT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RT_OK 0
#define RT_EINVAL (-1)   /* bad argument (NULL, non-positive size, grid not divisible by block, angle) */
#define RT_ENOMEM (-2)   /* device allocation failed */
#define RT_ECUDA (-3)    /* a CUDA call or kernel failed; see rt_last_error */
#define RT_EOPTICS (-4)  /* rt_set_optics: a field value is outside its physical range */
#define RT_ESTATE (-5)   /* a call before the call it needs: rt_trace before rt_set_optics, slots before rt_set_slots, ... */

#define RT_W0 (1ll << 32) /* tally quanta per photon */

/* Photon fates stored in records. */
#define RT_FATE_ATM_ABS 1
#define RT_FATE_SFC_ABS 2
#define RT_FATE_TOD_EXIT 3
#define RT_FATE_CAPPED 4
#define RT_FATE_ROULETTE 5 /* weighted mode only */

typedef struct rt_ctx rt_ctx; /* opaque; owned by the library; one CUDA device per context.  The calls on one
                                 context must be ordered (one stream, or streams synchronised by the caller):
                                 its launches share a work counter.  Use one context per concurrent stream. */

/* Always-on event counters, accumulated across rt_trace calls until rt_reset_tallies.
 * n_events = tentative collisions (null + real) = n_null + n_rayleigh + n_hg + n_atm_abs:
 * the "collision events" of BASELINE.json's metric. */
typedef struct {
  uint64_t n_photons, n_events, n_null, n_rayleigh, n_hg, n_atm_abs, n_sfc_hits, n_sfc_abs, n_toa,
      n_capped, n_cell_steps, n_relevel, n_roulette_killed, n_roulette_kept;
  int64_t capped_energy;   /* quanta of photons stopped by the event cap; 0 on all shipped configs */
  int64_t roulette_lost;   /* weighted mode: quanta of photons ended by the roulette ... */
  int64_t roulette_gained; /* ... and quanta given to its survivors (weight reset to RT_W0) */
} rt_counters;

/* Allocate a context for an nx*ny*nz grid of dx*dy*dz metre voxels with an acceleration grid
 * of bx*by*bz-voxel blocks ("coarser resolution than the simulation"; Q1).
 * nx,ny,nz must be multiples of bx,by,bz; bx*by*bz <= 4096; nx*ny*nz < 2^32.  Allocates packed optics
 * (16 B/voxel), the majorant grid and zeroed int64 tallies on cuda_device.  *out is owned
 * by the library until rt_destroy. */
int rt_create_grid(rt_ctx** out, int nx, int ny, int nz, float dx, float dy, float dz, int bx, int by,
                   int bz, int cuda_device);

/* Set the optical properties of one spectral point (k_ext, k_ext,cloud, omega0, g as 3D
 * fields; P:56 local surface albedo).  All five are owned by the caller, fp32, nvox / nvox / nvox /
 * nvox / ncol elements, each a DEVICE pointer (read in place) or a HOST pointer (detected; copied to a
 * device staging buffer on the stream first -- pinned memory makes that copy asynchronous).  They are
 * read on `cuda_stream` (a cudaStream_t, NULL = default stream) and may be freed once this call returns
 * (it synchronises the stream).  Packs cumulative
 * coefficients and builds the majorant grid (§3.5).  Validates k_ext >= 0 and
 * finite, 0 <= k_ext_cloud <= k_ext, 0 <= ssa <= 1, |g| < 1, 0 <= albedo <= 1 on the device;
 * a violation returns RT_EOPTICS (this call synchronises the stream to learn it). */
int rt_set_optics(rt_ctx* ctx, const float* k_ext, const float* k_ext_cloud, const float* ssa,
                  const float* g, const float* sfc_albedo, void* cuda_stream);

/* Trace n_photons photons with global ids first_photon_id .. first_photon_id + n_photons - 1
 * (DESIGN.md §3.6-3.12).  Sun at zenith_deg in [0, 90) and azimuth_deg clockwise from
 * north (position of the sun).  Random numbers: Philox4x32-10, key = seed, counter =
 * (photon id, event index, stream_id).  ADDS to the tallies and counters.  Asynchronous on
 * `cuda_stream`.  A call of more than 2^31 photons runs as consecutive launches of 2^31 (same photons: the parts are
 * index ranges of the one job); rt_trace_batch takes at most 2^31 photons per call. */
int rt_trace(rt_ctx* ctx, double zenith_deg, double azimuth_deg, uint64_t n_photons,
             uint64_t first_photon_id, uint64_t seed, uint32_t stream_id, void* cuda_stream);

/* As rt_trace, and also writes one 16-byte record per photon to records_out (DEVICE pointer,
 * 4 uint32 per photon, index = photon id - first_photon_id): word 0 = fate | surface hits << 8,
 * word 1 = terminal voxel or column index, word 2 = collision events, word 3 = real scatters. */
int rt_trace_records(rt_ctx* ctx, double zenith_deg, double azimuth_deg, uint64_t n_photons,
                     uint64_t first_photon_id, uint64_t seed, uint32_t stream_id, void* cuda_stream,
                     uint32_t* records_out);

/* A PART of a job (multi-GPU sharding; checkpointing): traces the photons with indices
 * [range_begin, range_begin + range_count) of the job that rt_trace(ctx, ..., job_photons, first_photon_id, ...)
 * would trace in one call -- same ids (first_photon_id + index), same columns and passes (§3.6 stratifies by
 * the index in the JOB), same Sobol shifts -- so the integer tallies of disjoint ranges covering
 * [0, job_photons), added up over calls, contexts or GPUs, equal the one-call tallies bit for bit.
 * records_out: NULL, or a DEVICE pointer to 16 B x range_count (index = job index - range_begin).
 * Errors: RT_EINVAL (range outside the job), else as rt_trace. */
int rt_trace_range(rt_ctx* ctx, double zenith_deg, double azimuth_deg, uint64_t job_photons,
                   uint64_t first_photon_id, uint64_t seed, uint32_t stream_id, void* cuda_stream,
                   uint64_t range_begin, uint64_t range_count, uint32_t* records_out);

/* Wait for the work THIS context has queued (on whichever streams its calls were given; other work on the
 * device is not waited for) and copy tallies out.  Each output may be a host or a
 * device pointer (detected), or NULL to skip: atm_abs nvox int64 in [z][y][x]; the others ncol
 * int64 in [y][x]; counters is a HOST pointer or NULL.  Energy closure: sum(atm_abs) +
 * sum(sfc_abs) + sum(toa_up) + capped_energy == n_photons * RT_W0 exactly. */
int rt_read_tallies(rt_ctx* ctx, int64_t* atm_abs, int64_t* sfc_dir, int64_t* sfc_dif, int64_t* sfc_abs,
                    int64_t* toa_up, rt_counters* counters);

/* rt_read_tallies without the wait: copies only, queued on `cuda_stream` after the work already queued there (the
 * counters go to pinned memory of the context as raw words and a host function queued on the stream,
 * cudaLaunchHostFunc, fills *counters from them: `counters` must be a HOST pointer; no kernel is launched, because
 * behind another context's persistent trace kernel a kernel of this stream would wait for that whole trace).  The
 * outputs are valid once the caller has synchronised that stream; at most two read-outs of one context may be in
 * flight.  HOST outputs should be pinned, or the copies serialise with the host.  Lets a caller upload the
 * next step's fields and download the last step's tallies while another context traces (bench.py's e2e leg). */
int rt_read_tallies_async(rt_ctx* ctx, int64_t* atm_abs, int64_t* sfc_dir, int64_t* sfc_dif, int64_t* sfc_abs,
                          int64_t* toa_up, rt_counters* counters, void* cuda_stream);

/* Merged acceleration cells (P:54 leaves the acceleration grid's resolution open).
 * Blocks of mx*my*mz acceleration cells in which the extinction is nearly uniform (max k_ext <=
 * merge_ratio * min k_ext over the block's voxels) are traversed as ONE cell with the block's maximum as
 * majorant: clear air above, below and between the clouds costs one step per block instead of one per
 * cell.  Any majorant >= k_ext gives the same expectations, so only the sample paths change.
 * mx, my, mz: powers of two, at most 64, dividing the acceleration grid's extents; 1,1,1 (the default after
 * rt_create_grid) = single-level grid.  merge_ratio >= 1.  Takes effect at the next rt_set_optics;
 * a context that already holds optics (in any slot) must be given them again before the next rt_trace or
 * rt_trace_batch: every majorant table was built for the old factors (RT_ESTATE otherwise).  Errors: RT_EINVAL. */
int rt_set_merge(rt_ctx* ctx, int mx, int my, int mz, float merge_ratio);

/* Absorption scheme of the following rt_trace calls.
 * RT_MODE_ANALOG (default; BASELINE.json north_star): a photon is absorbed with probability c1 / k_hat at a
 * tentative collision and (1 - albedo) at the surface, and ends in exactly one bin with RT_W0 quanta.
 * RT_MODE_WEIGHTED (the paper's scheme): the photon carries an integer weight w (RT_W0
 * at launch); every tentative collision deposits floor(w pq / 2^24) quanta in atm_abs[voxel], pq =
 * floor(c1 / k_hat 2^24), and continues with the rest; a surface arrival adds w to sfc_dir/sfc_dif, the
 * albedo splits it into sfc_abs and the reflected weight; a photon leaving through the top adds w to toa_up;
 * below RT_W0 / 2 the photon survives with probability w / RT_W0 and weight RT_W0, else it ends (fate 5).
 * Closure: sum(atm_abs) + sum(sfc_abs) + sum(toa_up) + capped_energy + roulette_lost - roulette_gained ==
 * n_photons * RT_W0 exactly.  Tallies of both modes may be accumulated in one context.  Errors: RT_EINVAL. */
#define RT_MODE_ANALOG 0
#define RT_MODE_WEIGHTED 1
int rt_set_mode(rt_ctx* ctx, int mode);

/* Top-of-domain source of the following rt_trace calls.  Default: every photon on the
 * sun beam, sub-pixel entry point from Philox (BASELINE.json north_star).
 * diffuse_fraction in [0, 1]: that share of the photons (decided per photon by a Philox word) starts diffuse:
 * direction drawn for isotropic downwelling radiance (pdf(mu) = 2 mu), counted as diffuse light from the start
 * ("the initial direction of each photon is either along the sun beam or randomly generated").
 * sampler RT_SAMPLER_SOBOL: within its column the photon of pass k (k = index in the call / ncol) enters at
 * point k of the 2-D Sobol sequence under a random digital shift per column, stream_id and first_photon_id
 * ("initialized ... following a scrambled Sobol sequence"); photons of the remainder pass keep Philox.
 * Errors: RT_EINVAL. */
#define RT_SAMPLER_PHILOX 0
#define RT_SAMPLER_SOBOL 1
int rt_set_source(rt_ctx* ctx, float diffuse_fraction, int sampler);

/* Batched spectral points (BASELINE.json configs[3]; "Ray tracing is then performed independently for each
 * quadrature point"): the context holds n_slots packed-optics, majorant and albedo slots in HBM (16 B per voxel
 * and slot: 112 points of the 512x512x128 grid = 57 GB of the B200's 180 GB), and ONE launch traces the photons
 * of all points, so that no launch drains between points and the host does not wait per point.
 * rt_set_slots: (re)allocates the slots (n_slots * nvox < 2^32; the 16 B x nvox records of the slots above 0 are
 *   allocated when the first of them is set); every slot must be given optics again afterwards.  Waits for the
 *   context's queued work.  Slot 0 is the one rt_set_optics writes and rt_trace reads; rt_trace itself needs
 *   rt_set_optics (which validates before returning): after rt_set_optics_slot(0), rt_set_optics_factored(0) or
 *   rt_set_point(0) slot 0 serves rt_trace_batch only and rt_trace returns RT_ESTATE until rt_set_optics is called.
 * rt_set_optics_slot: rt_set_optics into slot `slot`, asynchronous on `cuda_stream`: range errors are kept per
 *   slot on the device (setting a slot again clears its mask) and the next rt_trace_batch that launches the slot
 *   reports them, naming it (RT_EOPTICS).  Host fields are accepted but make the call wait for the stream.
 * rt_trace_batch: point j (first_point <= j < first_point + n_points <= n_slots) is traced with
 *   counts[j - first_point] photons (HOST array), stream id j, slot j, global photon ids first_photon_id + (index within the point), its own column stratification
 *   (full passes over the columns + remainder), i.e. exactly what rt_trace(..., counts[j], first_photon_id, seed,
 *   stream_id = j) on slot j's optics would trace; tallies accumulate.  records_out: NULL or 16 B per photon in
 *   the order of the points.  Reads the error mask and uploads the offsets before launching (waits for the
 *   stream once).  Errors: RT_EINVAL, RT_ESTATE (a slot without optics), RT_EOPTICS, RT_ENOMEM, RT_ECUDA. */
int rt_set_slots(rt_ctx* ctx, int n_slots);
int rt_set_optics_slot(rt_ctx* ctx, int slot, const float* k_ext, const float* k_ext_cloud, const float* ssa,
                       const float* g, const float* sfc_albedo, void* cuda_stream);
/* rt_set_optics_slot from FACTORED inputs (per spectral point the gas part of the optics depends on height
 * only; NEXT-3 of SURVEY.md §8(f)).  Per voxel at level z, in fp32 and in this order:
 *   k_ext = (k_abs[z] + k_ray[z]) + k_cloud;  ssa = (k_ray[z] + cloud_ssa * k_cloud) / k_ext (0 if k_ext = 0);
 *   k_ext_cloud = k_cloud;  g = cloud_g;  then packing and majorant exactly as rt_set_optics.
 * k_cloud ([z][y][x], nvox) and sfc_albedo (ncol) are DEVICE pointers (the cloud field is shared by all points
 * and uploaded once); k_abs, k_ray (nz each) may be HOST or DEVICE.  Reads 4 B per voxel instead of 16 and
 * needs 2 nz numbers per point from the host.  Asynchronous like rt_set_optics_slot (errors of the field values
 * at the next rt_trace_batch).  Requires rt_set_slots beforehand (RT_ESTATE), nx % 4 == 0, bx in {1, 2, 4},
 * by * bz <= 64.  Errors: RT_EINVAL, RT_ESTATE, RT_EOPTICS (cloud_ssa, cloud_g out of range), RT_ENOMEM, RT_ECUDA. */
int rt_set_optics_factored(rt_ctx* ctx, int slot, const float* k_cloud, const float* k_abs, const float* k_ray,
                           float cloud_ssa, float cloud_g, const float* sfc_albedo, void* cuda_stream);
/* Factored optics kept factored in the trace as well (NEXT-3 in full).  rt_set_cloud stores the cloud extinction
 * field once (own copy; DEVICE or HOST pointer; synchronises the stream to report a bad value, RT_EOPTICS) and
 * derives, per acceleration cell and level, its extrema.  rt_set_point then defines slot `slot` by the factors of
 * rt_set_optics_factored WITHOUT packing a 16-byte record per voxel: it only builds the point's majorant table
 * from those extrema (exact: fl(gas + k_cloud) is monotone in k_cloud) and keeps the 2 nz + 2 numbers; a
 * rt_trace_batch over such slots gathers 4 B of cloud extinction per tentative collision and rebuilds the
 * record of §3.4b + §3.4 with the same fp32 operations, so its photons are bit-identical to those of the packed
 * slots.  k_abs, k_ray (nz), sfc_albedo (ncol): HOST or DEVICE.  Needs rt_set_slots (any n >= 1) beforehand; the
 * points of one rt_trace_batch launch must all be of the same kind.  Per point this costs a pass over the cell
 * tables (a few MB) instead of over the voxel fields, and no 16 B x nvox slot.  Errors: RT_EINVAL, RT_ESTATE
 * (rt_set_point before rt_set_cloud), RT_EOPTICS, RT_ENOMEM, RT_ECUDA.
 * Voxel-sized acceleration cells (bx = by = bz = 1) with merging on (rt_set_merge): no majorant
 *   table is built per point at all.  A voxel-sized cell's majorant IS the voxel's extinction
 *   fl((k_abs[z] + k_ray[z]) + k_cloud), which the trace reads from the shared cloud field; rt_set_cloud derives the
 *   cloud extrema per block of mx x my x mz cells and level, and a point keeps one word per block (merged or not,
 *   and the block's maximum) plus nz gas sums.  Photons are bit-identical to those traced with the table
 *   (rt_set_optics_slot on the assembled fields).  In this mode rt_read_majorant returns RT_ESTATE after
 *   rt_set_point(0), and rt_set_merge also invalidates the cloud field (call rt_set_cloud again).
 * rt_set_points: the slots first_slot .. first_slot + n_points - 1 in one call.  k_abs, k_ray: [n_points][nz], HOST or
 *   DEVICE; cloud_ssa, cloud_g: HOST arrays of n_points; point p's albedo at sfc_albedo + p * albedo_stride (HOST or
 *   DEVICE; albedo_stride = 0: one albedo for all points, else >= ncol).  Same result as n_points rt_set_point calls;
 *   on voxel-sized merged cells it costs a fixed number of copies and two kernels whatever n_points is (the host's
 *   per-point call overhead is what a sweep over 112 points otherwise spends a tenth of its time on). */
int rt_set_cloud(rt_ctx* ctx, const float* k_cloud, void* cuda_stream);
int rt_set_point(rt_ctx* ctx, int slot, const float* k_abs, const float* k_ray, float cloud_ssa, float cloud_g,
                 const float* sfc_albedo, void* cuda_stream);
int rt_set_points(rt_ctx* ctx, int first_slot, int n_points, const float* k_abs, const float* k_ray,
                  const float* cloud_ssa, const float* cloud_g, const float* sfc_albedo, uint64_t albedo_stride,
                  void* cuda_stream);
int rt_trace_batch(rt_ctx* ctx, double zenith_deg, double azimuth_deg, int first_point, int n_points,
                   const uint64_t* counts, uint64_t first_photon_id, uint64_t seed, void* cuda_stream,
                   uint32_t* records_out);

/* Direct part of the heating (P:82 reports heating by direct and by diffuse radiation).  With on != 0 the
 * following rt_trace calls also add every quantum that a never-scattered photon deposits in atm_abs to a
 * second nvox-word tally (allocated at the first call, zeroed by rt_reset_tallies); atm_abs stays the total,
 * the diffuse part is the difference.  rt_read_heating_direct copies it out ([z][y][x], DEVICE or HOST
 * pointer) and synchronises.  Errors: RT_EINVAL, RT_ENOMEM, RT_ESTATE (read before enabling). */
int rt_set_heating_split(rt_ctx* ctx, int on);
int rt_read_heating_direct(rt_ctx* ctx, int64_t* atm_abs_direct);

/* S11, host helper ("The mean weight of all rays hitting the surface or leaving the domain top is then used
 * to compute surface and TOD radiative fluxes"; heating from the absorbed weight).  Converts `count` tally
 * quanta (HOST pointer, as read by rt_read_tallies) to physical units in double: every photon of the
 * n_photons traced into these tallies carries tod_flux * (domain area) / n_photons watts, where tod_flux is the
 * downward flux through the horizontal domain top in W m^-2 (the paper takes it from a two-stream
 * pre-computation, out of scope), so out[i] = tally[i] / RT_W0 * tod_flux * ncol / n_photons [W m^-2 per
 * column], divided by `depth` (the voxel depth dz in metres) when depth > 0 [W m^-3 for atm_abs].
 * Errors: RT_EINVAL (NULL, n_photons = 0, negative or non-finite arguments).  Runs on the host. */
int rt_tally_to_flux(const int64_t* tally, double* out, uint64_t count, uint64_t n_photons, uint64_t ncol,
                     double tod_flux, double depth);

/* Zero tallies and counters on `cuda_stream`. */
int rt_reset_tallies(rt_ctx* ctx, void* cuda_stream);

/* Copy the majorant grid ([cz][cy][cx] fp32, DEVICE or HOST pointer) out; for tests.  Cells of a merged
 * block hold -(block maximum) (sign bit set), the others their own maximum. */
int rt_read_majorant(rt_ctx* ctx, float* khat_out);

/* Copy the packed per-voxel coefficients (c1,c2,c3,g; 4 fp32 per voxel, [z][y][x]) out; for tests. */
int rt_read_packed_optics(rt_ctx* ctx, float* packed_out);

/* Random-gather microbenchmark for the roofline denominator: every thread issues
 * `loads_per_thread` independent 16-byte loads at Philox-random voxel indices among the first
 * `footprint_voxels` records of the context's packed-optics array (0 = the whole array; a footprint of
 * a few MiB measures L2, hundreds of MiB measures HBM).  Runs once untimed, then writes the elapsed
 * milliseconds of a second run (CUDA events on `cuda_stream`) to *ms_out and the number of 16-byte loads
 * issued to *n_loads_out.  Synchronises the stream. */
int rt_gather_bench(rt_ctx* ctx, uint32_t loads_per_thread, uint64_t footprint_voxels, void* cuda_stream,
                    float* ms_out, uint64_t* n_loads_out);

/* Milliseconds spent in the trace kernel of the most recent rt_trace* call on this context, from
 * CUDA events recorded on that call's stream around the launch.  Synchronises on the end event. */
int rt_last_trace_ms(rt_ctx* ctx, float* ms_out);

/* Kernel launches issued by this context so far (the library's own count). */
uint64_t rt_launch_count(const rt_ctx* ctx);

/* Philox4x32-10 words for n counters (DEVICE pointers: ctr n*4 uint32, out n*4 uint32); for the
 * bit-for-bit stream test. */
int rt_philox_words(int cuda_device, const uint32_t* ctr, uint32_t key0, uint32_t key1, uint32_t* out,
                    uint64_t n);

/* Self-test of the two places where the kernels replace an IEEE fp32 operation by the instruction sequence the compiler
 * itself uses on the fast side of that operation's range check (rt_device.cuh: rcp_in_range for 1 / x, sqrt_in_range
 * for sqrt(x); the operands there cannot leave the range): compares them with 1.0f / x and sqrtf(x)
 * over EVERY float of their ranges (reciprocal: 2^-126 <= |x| < 2^125, both signs; root: 2^-101 <= x <= FLT_MAX) and
 * writes the numbers of differing results, which must be 0 for the kernels to follow the stream definition bit for bit.
 * About 0.1 s.  Errors: RT_EINVAL, RT_ENOMEM, RT_ECUDA. */
int rt_selftest_ieee(int cuda_device, uint64_t* rcp_mismatches, uint64_t* sqrt_mismatches);

/* The majorant table WITHOUT any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Computes what rt_set_optics + rt_read_majorant give for the same
 * extinction field (the maximum of the extinction over each acceleration cell, and the merged
 * cells of §3.5b: every cell of a merged block holds -(block maximum)), bit for bit, with no context:
 *   k_ext    DEVICE, [z][y][x], nx * ny * nz floats (the total extinction, i.e. c3 of §3.4), read only;
 *   khat_out DEVICE, [cz][cy][cx], (nx/bx) * (ny/by) * (nz/bz) floats, written;
 *   bad_out  DEVICE int or NULL: set to 0, then to 1 if a value of k_ext is negative, NaN or infinite (the table is
 *            then unspecified); nothing is read back, so the call never waits for the GPU;
 *   mx, my, mz, merge_ratio as rt_set_merge (1, 1, 1 = no merging); cuda_device, cuda_stream: where it runs.
 * The per-cell minima the merge criterion needs are SCRATCH: they live in a file-scope device array of
 * RT_NO_ALLOC_MAX_CELLS floats (4 MiB, held by every GPU that loads the library until the process exits), so the cell
 * count must not exceed RT_NO_ALLOC_MAX_CELLS (RT_EINVAL, message via rt_no_alloc_last_error).  The call issues one
 * memset (bad_out) and two kernels on the stream and calls no cudaMalloc, cudaFree or other allocating routine.  All
 * calls on a device share that array: every call overwrites the part it reads before reading it (stale contents of an
 * earlier call never matter), but two calls that OVERLAP on the GPU (different streams, no dependency) race on it
 * and give wrong tables; put them on one stream or order them with events.
 * Errors: RT_EINVAL (NULL pointer, sizes, factors not powers of two dividing the cell grid, too many cells),
 * RT_ECUDA.  rt_no_alloc_last_error: the message of this thread's last failed rt_majorant_no_alloc call (never NULL). */
#define RT_NO_ALLOC_MAX_CELLS (1u << 20)
int rt_majorant_no_alloc(const float* k_ext, float* khat_out, int* bad_out, int nx, int ny, int nz, int bx, int by,
                         int bz, int mx, int my, int mz, float merge_ratio, int cuda_device, void* cuda_stream);
const char* rt_no_alloc_last_error(void);

const char* rt_last_error(const rt_ctx* ctx); /* never NULL; valid until the next call on ctx */
void rt_destroy(rt_ctx* ctx);                 /* frees all device memory; NULL is a no-op */

#ifdef __cplusplus
}
#endif
#endif
