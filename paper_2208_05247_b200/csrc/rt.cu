// rt.cu — C ABI of the photon tracer (include/rt.h) over the sm_100a kernels in rt_*.cuh.
// Host logic only: argument checks, device memory, launches.  No step of the method runs on the CPU.
#include "../../include/rt.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <utility>
#include <vector>

#include "rt_setup.cuh"
#include "rt_trace.cuh"

struct rt_ctx {
  int device = 0;
  int nx = 0, ny = 0, nz = 0, bx = 0, by = 0, bz = 0, ncx = 0, ncy = 0, ncz = 0;
  float dx = 0, dy = 0, dz = 0;
  int mx = 1, my = 1, mz = 1;             // merged-cell factors (rt_set_merge)
  float merge_ratio = 1.25f;
  int n_slots = 1;                        // rt_set_slots: optics / majorant / albedo slots (spectral points)
  std::vector<char> slot_ok = std::vector<char>(1, 0);
  // rt_read_tallies_async: the raw counter words are copied to pinned host memory and a host function queued on the
  // stream fills the caller's rt_counters from them (two buffers, used alternately: two read-outs may be in flight)
  struct CounterJob { unsigned long long raw[rt::C_COUNT]; rt_counters* out; };
  CounterJob* counter_jobs = nullptr;
  unsigned counter_calls = 0;
  int optics_slots = 1;                   // slots the packed-optics array currently holds (grown on demand)
  float* cloud = nullptr;                 // rt_set_cloud: own copy of the cloud field, nvox
  float* cloud_max = nullptr;             // ... highest / lowest cloud extinction per cell and level-in-cell
  float* cloud_min = nullptr;
  float2* point_par = nullptr;            // rt_set_point: (cloud_ssa, cloud_g) per slot
  bool cloud_ok = false;
  // voxel-sized cells + merging with the optics kept factored ("fly"): no majorant table per point;
  // per cloud field the extrema per block of merged cells and level ([block][mz]), per point one word per block and
  // the gas sums per level
  float* blk_max = nullptr;
  float* blk_min = nullptr;
  float* blk_tab = nullptr;               // [slot][block]: -(block maximum) if merged, else +maximum
  float* gas_sum = nullptr;               // [slot][nz]: fl(k_abs + k_ray)
  size_t blk_cap = 0;                     // floats blk_max / blk_min were allocated for
  int khat_slots = 1;                     // slots the majorant array currently holds (grown on demand, like optics)
  float* gas_tab = nullptr;               // rt_set_optics_factored: per slot k_abs[nz] then k_ray[nz] (device)
  unsigned batch_calls = 0;
  unsigned long long* batch_tab = nullptr; // device: offsets (n_slots + 1) then nfull (n_slots), for rt_trace_batch
  int weighted = 0;                       // rt_set_mode: 0 analog absorption, 1 weights + roulette
  float diffuse_fraction = 0.0f;          // rt_set_source
  int sobol = 0;
  unsigned long long* atm_dir = nullptr;  // rt_set_heating_split: heating by never-scattered photons, nvox words
  bool split = false;
  float* kmin = nullptr;                  // per-cell minimum extinction; allocated when merging is on
  size_t nvox = 0, ncol = 0, ncell = 0;
  float4* optics = nullptr;
  float* khat = nullptr;
  float* albedo = nullptr;
  unsigned long long* tallies = nullptr;  // atm_abs | sfc_dir | sfc_dif | sfc_abs | toa_up
  unsigned long long* counters = nullptr; // C_COUNT words, then the work counter
  int* bad = nullptr;                     // range-error masks on the device: one word per slot, then one for rt_set_cloud
  float* sink = nullptr;
  float* stage = nullptr;                 // 4 nvox + ncol floats; only allocated when a caller passes host fields
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  bool have_optics = false, have_trace = false;
  int trace_blocks[16] = {};              // persistent grid size per kernel instantiation [records | pow2 | weighted | batch]; 0 = not asked yet
  // streams this context has queued work on since the last wait, each with an event recorded after the latest
  // piece of work: rt_read_tallies waits for these instead of the whole device
  std::vector<std::pair<cudaStream_t, cudaEvent_t>> pending;
  cudaStream_t copy_stream = nullptr;     // non-blocking stream of the synchronous read-outs
  int sm_count = 0;
  uint64_t launches = 0;
  std::string err;
};

namespace {

struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int fail(rt_ctx* c, int code, const char* what, cudaError_t ce = cudaSuccess) {
  if (c) {
    c->err = what;
    if (ce != cudaSuccess) { c->err += ": "; c->err += cudaGetErrorString(ce); }
  }
  return code;
}

#define RT_CUDA(ctx, call)                                              \
  do {                                                                  \
    cudaError_t ce_ = (call);                                           \
    if (ce_ != cudaSuccess) return fail(ctx, ce_ == cudaErrorMemoryAllocation ? RT_ENOMEM : RT_ECUDA, #call, ce_); \
  } while (0)

void fill_counters(const unsigned long long* h, rt_counters* out) {
  out->n_null = h[rt::C_NULL]; out->n_rayleigh = h[rt::C_RAY]; out->n_hg = h[rt::C_HG];
  out->n_atm_abs = h[rt::C_ATM_ABS]; out->n_sfc_hits = h[rt::C_SFC_HITS];
  out->n_sfc_abs = h[rt::C_SFC_ABS]; out->n_toa = h[rt::C_TOA]; out->n_capped = h[rt::C_CAPPED];
  out->n_cell_steps = h[rt::C_CELLS]; out->n_relevel = h[rt::C_RELEVEL];
  out->n_roulette_killed = h[rt::C_ROUL_KILLED]; out->n_roulette_kept = h[rt::C_ROUL_KEPT];
  out->roulette_lost = (int64_t)h[rt::C_ROUL_LOST]; out->roulette_gained = (int64_t)h[rt::C_ROUL_GAINED];
  out->capped_energy = (int64_t)h[rt::C_CAPPED_E];
  out->n_events = h[rt::C_NULL] + h[rt::C_RAY] + h[rt::C_HG] + h[rt::C_ATM_ABS];
  out->n_photons = h[rt::C_ATM_ABS] + h[rt::C_SFC_ABS] + h[rt::C_TOA] + h[rt::C_CAPPED] + h[rt::C_ROUL_KILLED];
}
// Queued with cudaLaunchHostFunc behind the copy of the raw words; runs on a driver thread, calls no CUDA function.
void CUDART_CB counters_host_fn(void* p) {
  auto* job = static_cast<rt_ctx::CounterJob*>(p);
  fill_counters(job->raw, job->out);
}

// Remember that `st` now carries work of this context (an event after it), for rt_read_tallies' wait.
int mark(rt_ctx* c, cudaStream_t st) {
  for (auto& p : c->pending)
    if (p.first == st) { RT_CUDA(c, cudaEventRecord(p.second, st)); return RT_OK; }
  cudaEvent_t ev = nullptr;
  RT_CUDA(c, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
  c->pending.emplace_back(st, ev);
  RT_CUDA(c, cudaEventRecord(ev, st));
  return RT_OK;
}
// Wait for everything this context has queued, on whichever streams (not for other work on the device).
int wait_pending(rt_ctx* c) {
  for (auto& p : c->pending) RT_CUDA(c, cudaEventSynchronize(p.second));
  return RT_OK;
}

unsigned long long* tally_ptr(rt_ctx* c, int which) {  // 0 atm_abs, 1..4 the column tallies
  return which == 0 ? c->tallies : c->tallies + c->nvox + (size_t)(which - 1) * c->ncol;
}

// rt_set_optics accepts host fields too: they are copied to a device staging buffer on the stream.
// Returns the device pointer to read from, or nullptr after recording an error.
const float* stage_input(rt_ctx* c, const float* p, size_t n, size_t slot_offset, cudaStream_t st, int* rc) {
  cudaPointerAttributes at;
  cudaError_t ce = cudaPointerGetAttributes(&at, p);
  if (ce != cudaSuccess) { cudaGetLastError(); at.type = cudaMemoryTypeUnregistered; }
  if (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) return p;
  if (!c->stage) {
    ce = cudaMalloc(&c->stage, (4 * c->nvox + c->ncol) * sizeof(float));
    if (ce != cudaSuccess) { *rc = fail(c, RT_ENOMEM, "rt_set_optics: staging buffer for host fields", ce); return nullptr; }
  }
  float* dst = c->stage + slot_offset;
  ce = cudaMemcpyAsync(dst, p, n * sizeof(float), cudaMemcpyHostToDevice, st);
  if (ce != cudaSuccess) { *rc = fail(c, RT_ECUDA, "rt_set_optics: host-to-device copy", ce); return nullptr; }
  return dst;
}

bool fly_mode(const rt_ctx* c) {          // rt_set_cloud / rt_set_point without majorant tables
  return c->bx == 1 && c->by == 1 && c->bz == 1 && c->mx * c->my * c->mz > 1;
}
size_t n_blocks(const rt_ctx* c) { return c->ncell / ((size_t)c->mx * c->my * c->mz); }

// One source, 16 instantiations: <records, power-of-two wrap, weighted, batch>.
const void* pick_kernel(int variant) {
  switch (variant) {
#define RT_CASE(v) case v: return (const void*)rt::trace_kernel<((v) & 1) != 0, ((v) & 2) != 0, ((v) & 4) != 0, ((v) & 8) != 0>;
    RT_CASE(0) RT_CASE(1) RT_CASE(2) RT_CASE(3) RT_CASE(4) RT_CASE(5) RT_CASE(6) RT_CASE(7)
    RT_CASE(8) RT_CASE(9) RT_CASE(10) RT_CASE(11) RT_CASE(12) RT_CASE(13) RT_CASE(14) RT_CASE(15)
#undef RT_CASE
  }
  return nullptr;
}
// Persistent grid of one instantiation: resident blocks per SM (occupancy query, once per instantiation) x SM count.
int trace_grid(rt_ctx* c, int variant, const void* fn, int* blocks_out) {
  int& cached = c->trace_blocks[variant];
  if (cached == 0) {
    int per_sm = 0;
    RT_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, rt::kTraceThreads, 0));
    if (per_sm < 1) return fail(c, RT_ECUDA, "rt_trace: the trace kernel does not fit on an SM");
    cached = c->sm_count * per_sm;
  }
  *blocks_out = cached;
  return RT_OK;
}

int do_trace(rt_ctx* c, double zenith_deg, double azimuth_deg, uint64_t n_photons, uint64_t first_id,
             uint64_t seed, uint32_t stream_id, void* stream_v, uint32_t* records, int n_points = 0, int first_point = 0,
             const unsigned long long* tab = nullptr, bool factored_trace = false, uint64_t index_base = 0,
             uint64_t job_photons = 0) {
  if (!c) return RT_EINVAL;
  if (job_photons == 0) job_photons = n_photons;   // a whole job in one call
  if (n_points == 0 && !c->have_optics) return fail(c, RT_ESTATE, "rt_trace: call rt_set_optics first");
  if (!(zenith_deg >= 0.0 && zenith_deg < 90.0) || !std::isfinite(azimuth_deg))
    return fail(c, RT_EINVAL, "rt_trace: zenith must be in [0, 90) degrees and azimuth finite");
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)stream_v;
  rt::TraceArgs A;
  A.nx = c->nx; A.ny = c->ny; A.nz = c->nz; A.bx = c->bx; A.by = c->by; A.bz = c->bz;
  A.ncx = c->ncx; A.ncy = c->ncy; A.ncz = c->ncz;
  A.dx = c->dx; A.dy = c->dy; A.dz = c->dz;
  A.rdx = 1.0f / c->dx; A.rdy = 1.0f / c->dy; A.rdz = 1.0f / c->dz;
  A.Lx = (float)c->bx * c->dx; A.Ly = (float)c->by * c->dy; A.Lz = (float)c->bz * c->dz;
  A.rLx = 1.0f / A.Lx; A.rLy = 1.0f / A.Ly; A.rLz = 1.0f / A.Lz;
  A.mx = c->mx; A.my = c->my; A.mz = c->mz;
  A.unit = (c->bx == 1 && c->by == 1 && c->bz == 1) ? 1 : 0;
  A.vote_bias = rt::vote_bias(A.unit ? rt::kCollideBatchUnit : rt::kCollideBatch);
  A.move_steps = A.unit ? rt::kMoveStepsUnit : rt::kMoveSteps;
  A.rmx = 1.0f / (float)c->mx; A.rmy = 1.0f / (float)c->my; A.rmz = 1.0f / (float)c->mz;
  A.Lx1 = (float)(c->mx * c->bx) * c->dx; A.Ly1 = (float)(c->my * c->by) * c->dy; A.Lz1 = (float)(c->mz * c->bz) * c->dz;
  // sun direction evaluated in double on the host, rounded once to fp32
  const double deg = 3.14159265358979323846 / 180.0;
  const double th = zenith_deg * deg, ph = azimuth_deg * deg;
  auto nudged = [](double d) { const float f = (float)d; return std::fabs(f) < rt::kTiny ? rt::kTiny : f; };   // Q20
  A.sun_x = nudged(-std::sin(th) * std::sin(ph));
  A.sun_y = nudged(-std::sin(th) * std::cos(ph));
  A.sun_z = nudged(-std::cos(th));
  A.sun_ix = 1.0f / A.sun_x; A.sun_iy = 1.0f / A.sun_y; A.sun_iz = 1.0f / A.sun_z;   // IEEE fp32, as place()
  A.optics = c->optics; A.khat = c->khat; A.albedo = c->albedo;
  A.atm_dir = c->split ? c->atm_dir : nullptr;
  A.atm_abs = tally_ptr(c, 0); A.sfc_dir = tally_ptr(c, 1); A.sfc_dif = tally_ptr(c, 2);
  A.sfc_abs = tally_ptr(c, 3); A.toa_up = tally_ptr(c, 4);
  A.counters = c->counters; A.next_photon = c->counters + rt::C_COUNT;
  A.records = records;
  A.n_photons = n_photons; A.first_id = first_id; A.ncol = c->ncol; A.index_base = index_base;
  A.n_full = (job_photons / c->ncol) * c->ncol;
  // the packed cell index of the kPow2 instantiations (rt_trace.cuh TraceArgs) needs every reachable index, one merged
  // step beyond the top included, below 2^31
  const bool pow2 = !(c->ncx & (c->ncx - 1)) && !(c->ncy & (c->ncy - 1)) &&
                    (unsigned long long)c->ncell + 64ull * c->ncx * c->ncy < (1ull << 31);
  if (pow2) {
    auto log2i = [](int v) { int l = 0; while ((1 << l) < v) ++l; return l; };
    A.lx = log2i(c->ncx); A.shz = A.lx + log2i(c->ncy);
    A.xmask = (unsigned)c->ncx - 1u; A.ymask = ((unsigned)c->ncy - 1u) << A.lx; A.zmask = ~((1u << A.shz) - 1u);
    A.omask = ~(((unsigned)c->mx - 1u) | (((unsigned)c->my - 1u) << A.lx) | (((unsigned)c->mz - 1u) << A.shz));
  } else {
    A.lx = A.shz = 0; A.xmask = A.ymask = A.zmask = A.omask = 0u;
  }
  const int variant = (records ? 1 : 0) | (pow2 ? 2 : 0) | (c->weighted ? 4 : 0) | (n_points > 0 ? 8 : 0);
  const void* fn = pick_kernel(variant);
  int blocks = 0;
  if (int rcg = trace_grid(c, variant, fn, &blocks)) return rcg;
  {
    // ids per work-counter atomic: 128, or fewer (a multiple of 32) when the launch has under ~8 chunks per warp,
    // so that short launches (one spectral point of config 4) balance over all resident warps
    const unsigned long long warps = (unsigned long long)blocks * (rt::kTraceThreads / 32);
    unsigned long long ch = n_photons / (warps * 8ull);
    ch = (ch / 32ull) * 32ull;
    A.chunk = (unsigned)(ch < 32ull ? 32ull : (ch > (unsigned long long)rt::kChunk ? (unsigned long long)rt::kChunk : ch));
  }
  A.keys = rt::philox_round_keys((uint32_t)seed, (uint32_t)(seed >> 32)); A.stream_id = stream_id;
  A.keys_sobol = rt::philox_round_keys((uint32_t)seed, (uint32_t)(seed >> 32) ^ 0x534F424Cu);
  A.diffuse_fraction = c->diffuse_fraction; A.sobol = c->sobol;
  A.n_points = n_points; A.first_point = first_point; A.offsets = tab; A.nfull = tab ? tab + c->n_slots + 1 : nullptr;
  A.nvox32 = (unsigned)c->nvox; A.ncell32 = (unsigned)c->ncell; A.ncol32 = (unsigned)c->ncol;
  A.cloud = factored_trace ? c->cloud : nullptr; A.gas = c->gas_tab; A.point_par = c->point_par;
  A.fly = (factored_trace && fly_mode(c)) ? 1 : 0;
  if (A.fly) A.move_steps = rt::kMoveStepsFly;
  A.btab = c->blk_tab; A.gsum = c->gas_sum;
  auto log2i = [](int v) { int l = 0; while ((1 << l) < v) ++l; return l; };
  A.lmx = log2i(c->mx); A.lmy = log2i(c->my); A.lmz = log2i(c->mz);
  A.nbx = c->ncx / c->mx; A.nby = c->ncy / c->my; A.nblk32 = (unsigned)n_blocks(c);
  RT_CUDA(c, cudaEventRecord(c->ev0, st));
  // one launch per 2^31 photons at most (the kernel counts a block's finished photons in 32-bit words); the parts
  // are consecutive index ranges of the same job, so photons and tallies do not depend on the split
  const unsigned long long kMaxLaunch = 1ull << 31;
  for (unsigned long long off = 0; off < n_photons; off += kMaxLaunch) {
    if (n_points > 0 && n_photons > kMaxLaunch) return fail(c, RT_EINVAL, "rt_trace_batch: at most 2^31 photons per launch");
    A.n_photons = n_photons - off < kMaxLaunch ? n_photons - off : kMaxLaunch;
    A.index_base = index_base + off;
    A.records = records ? records + 4ull * off : nullptr;
    RT_CUDA(c, cudaMemsetAsync(A.next_photon, 0, sizeof(unsigned long long), st));
    void* kargs[1] = {(void*)&A};
    RT_CUDA(c, cudaLaunchKernel(fn, dim3((unsigned)blocks), dim3((unsigned)rt::kTraceThreads), kargs, 0, st));
    ++c->launches;
  }
  RT_CUDA(c, cudaEventRecord(c->ev1, st));
  RT_CUDA(c, cudaGetLastError());
  c->have_trace = true;
  return mark(c, st);
}

}  // namespace

extern "C" {

int rt_create_grid(rt_ctx** out, int nx, int ny, int nz, float dx, float dy, float dz, int bx, int by,
                   int bz, int cuda_device) {
  if (!out) return RT_EINVAL;
  *out = nullptr;
  if (nx <= 0 || ny <= 0 || nz <= 0 || bx <= 0 || by <= 0 || bz <= 0) return RT_EINVAL;
  if (nx % bx || ny % by || nz % bz || (long long)bx * by * bz > 4096) return RT_EINVAL;
  if (!(dx > 0.0f) || !(dy > 0.0f) || !(dz > 0.0f)) return RT_EINVAL;
  if ((unsigned long long)nx * ny * nz >= (1ull << 32)) return RT_EINVAL;   // voxel indices are 32-bit in the kernels
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) return RT_ECUDA;
  rt_ctx* c = new rt_ctx();
  c->device = cuda_device;
  c->nx = nx; c->ny = ny; c->nz = nz; c->bx = bx; c->by = by; c->bz = bz;
  c->ncx = nx / bx; c->ncy = ny / by; c->ncz = nz / bz;
  c->dx = dx; c->dy = dy; c->dz = dz;
  c->nvox = (size_t)nx * ny * nz; c->ncol = (size_t)nx * ny; c->ncell = (size_t)c->ncx * c->ncy * c->ncz;
  *out = c;  // returned even on failure so rt_last_error works; caller still calls rt_destroy
  DeviceGuard guard(cuda_device);
  const size_t ntally = c->nvox + 4 * c->ncol;
  RT_CUDA(c, cudaMalloc(&c->optics, c->nvox * sizeof(float4)));
  RT_CUDA(c, cudaMalloc(&c->khat, c->ncell * sizeof(float)));
  RT_CUDA(c, cudaMalloc(&c->albedo, c->ncol * sizeof(float)));
  RT_CUDA(c, cudaMalloc(&c->tallies, ntally * sizeof(unsigned long long)));
  RT_CUDA(c, cudaMalloc(&c->counters, (rt::C_COUNT + 1) * sizeof(unsigned long long)));
  RT_CUDA(c, cudaMalloc(&c->bad, 2 * sizeof(int)));
  RT_CUDA(c, cudaMemset(c->bad, 0, 2 * sizeof(int)));
  RT_CUDA(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
  RT_CUDA(c, cudaMalloc(&c->sink, sizeof(float)));
  RT_CUDA(c, cudaMemset(c->tallies, 0, ntally * sizeof(unsigned long long)));
  RT_CUDA(c, cudaMemset(c->counters, 0, (rt::C_COUNT + 1) * sizeof(unsigned long long)));
  RT_CUDA(c, cudaEventCreate(&c->ev0));
  RT_CUDA(c, cudaEventCreate(&c->ev1));
  RT_CUDA(c, cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, cuda_device));
  return RT_OK;
}

}  // extern "C" (reopened below)

namespace {

// The packed-optics array holds one slot until a packed slot > 0 is asked for; then it is grown to all n_slots
// (16 B per voxel and slot), keeping what it holds.
int ensure_khat_slots(rt_ctx* c, int slot) {
  if (slot < c->khat_slots) return RT_OK;
  DeviceGuard guard(c->device);
  if (int rcw = wait_pending(c)) return rcw;
  float* grown = nullptr;
  RT_CUDA(c, cudaMalloc(&grown, (size_t)c->n_slots * c->ncell * sizeof(float)));
  RT_CUDA(c, cudaMemcpy(grown, c->khat, (size_t)c->khat_slots * c->ncell * sizeof(float), cudaMemcpyDeviceToDevice));
  cudaFree(c->khat);
  c->khat = grown;
  c->khat_slots = c->n_slots;
  return RT_OK;
}

int ensure_optics_slots(rt_ctx* c, int slot) {
  if (slot < c->optics_slots) return RT_OK;
  DeviceGuard guard(c->device);
  if (int rcw = wait_pending(c)) return rcw;
  float4* grown = nullptr;
  RT_CUDA(c, cudaMalloc(&grown, (size_t)c->n_slots * c->nvox * sizeof(float4)));
  RT_CUDA(c, cudaMemcpy(grown, c->optics, (size_t)c->optics_slots * c->nvox * sizeof(float4), cudaMemcpyDeviceToDevice));
  cudaFree(c->optics);
  c->optics = grown;
  c->optics_slots = c->n_slots;
  return RT_OK;
}

// S0 + S1 into optics / majorant / albedo slot `slot`.  Range errors go to the slot's own mask word (cleared here,
// so re-setting a slot with good data heals it).  sync: wait for the kernels and report the mask now
// (rt_set_optics); otherwise rt_trace_batch reads the masks of the slots it launches.
int set_optics_impl(rt_ctx* c, int slot, const float* k_ext, const float* k_ext_cloud, const float* ssa,
                    const float* g, const float* sfc_albedo, cudaStream_t st, bool sync, const char* who) {
  if (!k_ext || !k_ext_cloud || !ssa || !g || !sfc_albedo) return fail(c, RT_EINVAL, "rt_set_optics: NULL field");
  DeviceGuard guard(c->device);
  if (int rce = ensure_optics_slots(c, slot)) return rce;
  if (int rce = ensure_khat_slots(c, slot)) return rce;
  c->slot_ok[slot] = 0;
  if (slot == 0) c->have_optics = false;
  int rc = RT_OK;
  const float* in[5] = {k_ext, k_ext_cloud, ssa, g, sfc_albedo};
  k_ext = stage_input(c, k_ext, c->nvox, 0, st, &rc);                      if (!k_ext) return rc;
  k_ext_cloud = stage_input(c, k_ext_cloud, c->nvox, c->nvox, st, &rc);    if (!k_ext_cloud) return rc;
  ssa = stage_input(c, ssa, c->nvox, 2 * c->nvox, st, &rc);                if (!ssa) return rc;
  g = stage_input(c, g, c->nvox, 3 * c->nvox, st, &rc);                    if (!g) return rc;
  sfc_albedo = stage_input(c, sfc_albedo, c->ncol, 4 * c->nvox, st, &rc);  if (!sfc_albedo) return rc;
  const bool staged = in[0] != k_ext || in[1] != k_ext_cloud || in[2] != ssa || in[3] != g || in[4] != sfc_albedo;
  float4* optics = c->optics + (size_t)slot * c->nvox;
  float* khat = c->khat + (size_t)slot * c->ncell;
  float* albedo = c->albedo + (size_t)slot * c->ncol;
  const bool rows = (c->nx % 4 == 0) && !(((uintptr_t)k_ext | (uintptr_t)k_ext_cloud | (uintptr_t)ssa | (uintptr_t)g) & 15u);
  const bool cellrows = rows && (c->bx == 1 || c->bx == 2 || c->bx == 4) && c->by * c->bz <= 64;   // no atomics, no zeroing
  int* bad = c->bad + slot;
  RT_CUDA(c, cudaMemsetAsync(bad, 0, sizeof(int), st));
  if (!cellrows) RT_CUDA(c, cudaMemsetAsync(khat, 0, c->ncell * sizeof(float), st));
  RT_CUDA(c, cudaMemcpyAsync(albedo, sfc_albedo, c->ncol * sizeof(float), cudaMemcpyDeviceToDevice, st));
  const int blocks = c->sm_count * 8;
  const bool merging = c->mx * c->my * c->mz > 1;
  if (merging) {
    if (!c->kmin) RT_CUDA(c, cudaMalloc(&c->kmin, c->ncell * sizeof(float)));
    if (!cellrows) RT_CUDA(c, cudaMemsetAsync(c->kmin, 0x7f, c->ncell * sizeof(float), st));   // 0x7f7f7f7f: above any finite input's bits that matter (3.4e38)
  }
  if (cellrows)
    rt::pack_optics_cellrows_kernel<<<c->sm_count * 16, 128, 0, st>>>(
        (const float4*)k_ext, (const float4*)k_ext_cloud, (const float4*)ssa, (const float4*)g, optics,
        khat, merging ? c->kmin : nullptr, c->nx, c->ny, c->nz, c->bx, c->by, c->bz, bad);
  else if (rows)
    rt::pack_optics_rows_kernel<<<c->sm_count * 16, 128, 0, st>>>(
        (const float4*)k_ext, (const float4*)k_ext_cloud, (const float4*)ssa, (const float4*)g, optics,
        (int*)khat, merging ? (int*)c->kmin : nullptr, c->nx, c->ny, c->nz, c->bx, c->by, c->bz, bad);
  else
    rt::pack_optics_kernel<<<blocks, 256, 0, st>>>(k_ext, k_ext_cloud, ssa, g, optics, (int*)khat,
                                                  merging ? (int*)c->kmin : nullptr, c->nx,
                                                  c->ny, c->nz, c->bx, c->by, c->bz, bad);
  rt::check_albedo_kernel<<<c->sm_count, 256, 0, st>>>(albedo, c->ncol, bad);
  c->launches += 2;
  if (merging) {
    const size_t nblk = c->ncell / ((size_t)c->mx * c->my * c->mz);
    rt::merge_cells_kernel<<<(unsigned)((nblk * 32 + 127) / 128), 128, 0, st>>>(khat, c->kmin, c->ncx, c->ncy, c->ncz,
                                                                            c->mx, c->my, c->mz, c->merge_ratio);
    ++c->launches;
  }
  RT_CUDA(c, cudaGetLastError());
  if (int rcm = mark(c, st)) return rcm;
  if (sync) {
    int hbad = 0;
    RT_CUDA(c, cudaMemcpyAsync(&hbad, bad, sizeof(int), cudaMemcpyDeviceToHost, st));
    RT_CUDA(c, cudaStreamSynchronize(st));
    if (hbad) {
      char msg[176];
      snprintf(msg, sizeof msg, "%s: input out of range (mask 0x%x: 1 k_ext, 2 k_ext_cloud, 4 ssa, 8 g, 16 albedo)", who, hbad);
      return fail(c, RT_EOPTICS, msg);
    }
  } else if (staged) {
    RT_CUDA(c, cudaStreamSynchronize(st));   // the one staging buffer is about to be reused
  }
  c->slot_ok[slot] = 1;
  if (slot == 0 && sync) c->have_optics = true;
  return RT_OK;
}

}  // namespace

extern "C" {

int rt_set_optics(rt_ctx* c, const float* k_ext, const float* k_ext_cloud, const float* ssa, const float* g,
                  const float* sfc_albedo, void* cuda_stream) {
  if (!c) return RT_EINVAL;
  return set_optics_impl(c, 0, k_ext, k_ext_cloud, ssa, g, sfc_albedo, (cudaStream_t)cuda_stream, true, "rt_set_optics");
}

int rt_set_slots(rt_ctx* c, int n_slots) {
  if (!c) return RT_EINVAL;
  if (n_slots < 1 || (unsigned long long)n_slots * c->nvox >= (1ull << 32))
    return fail(c, RT_EINVAL, "rt_set_slots: need 1 <= n_slots and n_slots * nvox < 2^32");
  DeviceGuard guard(c->device);
  if (int rcw = wait_pending(c)) return rcw;
  cudaFree(c->optics); cudaFree(c->khat); cudaFree(c->albedo); cudaFree(c->batch_tab); cudaFree(c->gas_tab); cudaFree(c->point_par); cudaFree(c->bad);
  cudaFree(c->blk_tab); cudaFree(c->gas_sum); c->blk_tab = nullptr; c->gas_sum = nullptr;
  c->optics = nullptr; c->khat = nullptr; c->albedo = nullptr; c->batch_tab = nullptr; c->gas_tab = nullptr; c->point_par = nullptr; c->bad = nullptr;
  c->have_optics = false;
  c->n_slots = n_slots;
  c->slot_ok.assign((size_t)n_slots, 0);
  RT_CUDA(c, cudaMalloc(&c->optics, c->nvox * sizeof(float4)));   // one slot; grown when a packed slot > 0 is set
  c->optics_slots = 1;
  RT_CUDA(c, cudaMalloc(&c->khat, c->ncell * sizeof(float)));     // one slot; grown when a slot > 0 needs a table
  c->khat_slots = 1;
  RT_CUDA(c, cudaMalloc(&c->albedo, (size_t)n_slots * c->ncol * sizeof(float)));
  RT_CUDA(c, cudaMalloc(&c->batch_tab, 2 * (2 * (size_t)n_slots + 1) * sizeof(unsigned long long)));   // two launches may be in flight
  RT_CUDA(c, cudaMalloc(&c->bad, ((size_t)n_slots + 1) * sizeof(int)));
  RT_CUDA(c, cudaMemset(c->bad, 0, ((size_t)n_slots + 1) * sizeof(int)));
  return RT_OK;
}

int rt_set_optics_slot(rt_ctx* c, int slot, const float* k_ext, const float* k_ext_cloud, const float* ssa,
                       const float* g, const float* sfc_albedo, void* cuda_stream) {
  if (!c) return RT_EINVAL;
  if (slot < 0 || slot >= c->n_slots) return fail(c, RT_EINVAL, "rt_set_optics_slot: slot out of range (rt_set_slots)");
  return set_optics_impl(c, slot, k_ext, k_ext_cloud, ssa, g, sfc_albedo, (cudaStream_t)cuda_stream, false,
                         "rt_set_optics_slot");
}

int rt_set_optics_factored(rt_ctx* c, int slot, const float* k_cloud, const float* k_abs, const float* k_ray,
                           float cloud_ssa, float cloud_g, const float* sfc_albedo, void* cuda_stream) {
  if (!c) return RT_EINVAL;
  if (slot < 0 || slot >= c->n_slots) return fail(c, RT_EINVAL, "rt_set_optics_factored: slot out of range (rt_set_slots)");
  if (!c->batch_tab) return fail(c, RT_ESTATE, "rt_set_optics_factored: call rt_set_slots first");
  if (!k_cloud || !k_abs || !k_ray || !sfc_albedo) return fail(c, RT_EINVAL, "rt_set_optics_factored: NULL argument");
  if (c->nx % 4 || !(c->bx == 1 || c->bx == 2 || c->bx == 4) || c->by * c->bz > 64 || ((uintptr_t)k_cloud & 15u))
    return fail(c, RT_EINVAL, "rt_set_optics_factored: needs nx % 4 == 0, bx in {1, 2, 4}, by * bz <= 64, 16-byte aligned k_cloud");
  if (!(cloud_ssa >= 0.0f && cloud_ssa <= 1.0f) || !(std::fabs(cloud_g) < 1.0f))
    return fail(c, RT_EOPTICS, "rt_set_optics_factored: cloud_ssa must be in [0, 1] and |cloud_g| < 1");
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  for (const void* p : {(const void*)k_cloud, (const void*)sfc_albedo}) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess || !(at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged)) {
      cudaGetLastError();
      return fail(c, RT_EINVAL, "rt_set_optics_factored: k_cloud and sfc_albedo must be device pointers");
    }
  }
  if (int rce = ensure_optics_slots(c, slot)) return rce;
  if (int rce = ensure_khat_slots(c, slot)) return rce;
  c->slot_ok[slot] = 0;
  if (slot == 0) c->have_optics = false;
  if (!c->gas_tab) RT_CUDA(c, cudaMalloc(&c->gas_tab, (size_t)c->n_slots * 2 * c->nz * sizeof(float)));
  float* tab = c->gas_tab + (size_t)slot * 2 * c->nz;
  RT_CUDA(c, cudaMemcpyAsync(tab, k_abs, c->nz * sizeof(float), cudaMemcpyDefault, st));
  RT_CUDA(c, cudaMemcpyAsync(tab + c->nz, k_ray, c->nz * sizeof(float), cudaMemcpyDefault, st));
  float4* optics = c->optics + (size_t)slot * c->nvox;
  float* khat = c->khat + (size_t)slot * c->ncell;
  float* albedo = c->albedo + (size_t)slot * c->ncol;
  RT_CUDA(c, cudaMemcpyAsync(albedo, sfc_albedo, c->ncol * sizeof(float), cudaMemcpyDeviceToDevice, st));
  const bool merging = c->mx * c->my * c->mz > 1;
  if (merging && !c->kmin) RT_CUDA(c, cudaMalloc(&c->kmin, c->ncell * sizeof(float)));
  RT_CUDA(c, cudaMemsetAsync(c->bad + slot, 0, sizeof(int), st));
  rt::pack_factored_cellrows_kernel<<<c->sm_count * 16, 128, 0, st>>>(
      (const float4*)k_cloud, tab, tab + c->nz, cloud_ssa, cloud_g, optics, khat, merging ? c->kmin : nullptr,
      c->nx, c->ny, c->nz, c->bx, c->by, c->bz, c->bad + slot);
  rt::check_albedo_kernel<<<c->sm_count, 256, 0, st>>>(albedo, c->ncol, c->bad + slot);
  c->launches += 2;
  if (merging) {
    const size_t nblk = c->ncell / ((size_t)c->mx * c->my * c->mz);
    rt::merge_cells_kernel<<<(unsigned)((nblk * 32 + 127) / 128), 128, 0, st>>>(khat, c->kmin, c->ncx, c->ncy, c->ncz,
                                                                                 c->mx, c->my, c->mz, c->merge_ratio);
    ++c->launches;
  }
  RT_CUDA(c, cudaGetLastError());
  c->slot_ok[slot] = 1;
  return mark(c, st);
}

int rt_set_cloud(rt_ctx* c, const float* k_cloud, void* cuda_stream) {
  if (!c || !k_cloud) return c ? fail(c, RT_EINVAL, "rt_set_cloud: NULL field") : RT_EINVAL;
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  c->cloud_ok = false;
  for (auto& ok : c->slot_ok) if (ok == 2) ok = 0;      // points built on the old cloud field
  if (!c->cloud) RT_CUDA(c, cudaMalloc(&c->cloud, c->nvox * sizeof(float)));
  const bool fly = fly_mode(c);
  if (fly) {
    const size_t need = n_blocks(c) * c->mz;                // sized by the merge factors
    if (need > c->blk_cap) {
      if (int rcw = wait_pending(c)) return rcw;
      cudaFree(c->blk_max); cudaFree(c->blk_min); c->blk_max = c->blk_min = nullptr; c->blk_cap = 0;
      RT_CUDA(c, cudaMalloc(&c->blk_max, need * sizeof(float)));
      RT_CUDA(c, cudaMalloc(&c->blk_min, need * sizeof(float)));
      c->blk_cap = need;
    }
  } else {
    if (!c->cloud_max) RT_CUDA(c, cudaMalloc(&c->cloud_max, c->ncell * c->bz * sizeof(float)));
    if (!c->cloud_min) RT_CUDA(c, cudaMalloc(&c->cloud_min, c->ncell * c->bz * sizeof(float)));
  }
  RT_CUDA(c, cudaMemcpyAsync(c->cloud, k_cloud, c->nvox * sizeof(float), cudaMemcpyDefault, st));
  int* cbad = c->bad + c->n_slots;        // the cloud field's own mask word: the slots' masks are not touched
  RT_CUDA(c, cudaMemsetAsync(cbad, 0, sizeof(int), st));
  if (fly)
    rt::cloud_blocks_kernel<<<(unsigned)((n_blocks(c) * 32 + 127) / 128), 128, 0, st>>>(
        c->cloud, c->blk_max, c->blk_min, c->nx, c->ny, c->nz, c->mx, c->my, c->mz, cbad);
  else
    rt::cloud_levels_kernel<<<c->sm_count * 8, 256, 0, st>>>(c->cloud, c->cloud_max, c->cloud_min, c->nx, c->ny, c->nz,
                                                             c->bx, c->by, c->bz, cbad);
  ++c->launches;
  RT_CUDA(c, cudaGetLastError());
  if (int rcm = mark(c, st)) return rcm;
  int bad = 0;
  RT_CUDA(c, cudaMemcpyAsync(&bad, cbad, sizeof(int), cudaMemcpyDeviceToHost, st));
  RT_CUDA(c, cudaStreamSynchronize(st));
  if (bad) return fail(c, RT_EOPTICS, "rt_set_cloud: the cloud extinction must be finite and >= 0");
  c->cloud_ok = true;
  return RT_OK;
}

// rt_set_point / rt_set_points on voxel-sized merged cells: the gas profiles, (cloud_ssa, cloud_g) and albedo of n
// consecutive slots with a fixed number of copies and two kernels, whatever n is.
static int set_points_fly(rt_ctx* c, int first, int n, const float* k_abs, const float* k_ray, const float* cloud_ssa,
                          const float* cloud_g, const float* sfc_albedo, uint64_t albedo_stride, cudaStream_t st) {
  const size_t nz = (size_t)c->nz, nblk = n_blocks(c);
  if (!c->blk_tab) RT_CUDA(c, cudaMalloc(&c->blk_tab, (size_t)c->n_slots * nblk * sizeof(float)));
  if (!c->gas_sum) RT_CUDA(c, cudaMalloc(&c->gas_sum, (size_t)c->n_slots * nz * sizeof(float)));
  float* tab = c->gas_tab + (size_t)first * 2 * nz;
  RT_CUDA(c, cudaMemcpy2DAsync(tab, 2 * nz * sizeof(float), k_abs, nz * sizeof(float), nz * sizeof(float), (size_t)n, cudaMemcpyDefault, st));
  RT_CUDA(c, cudaMemcpy2DAsync(tab + nz, 2 * nz * sizeof(float), k_ray, nz * sizeof(float), nz * sizeof(float), (size_t)n, cudaMemcpyDefault, st));
  std::vector<float2> pp((size_t)n);
  for (int p = 0; p < n; ++p) pp[(size_t)p] = make_float2(cloud_ssa[p], cloud_g[p]);
  RT_CUDA(c, cudaMemcpyAsync(c->point_par + first, pp.data(), (size_t)n * sizeof(float2), cudaMemcpyHostToDevice, st));   // pageable: staged before return
  float* albedo = c->albedo + (size_t)first * c->ncol;
  const bool broadcast = n > 1 && albedo_stride == 0;
  if (broadcast || n == 1)
    RT_CUDA(c, cudaMemcpyAsync(albedo, sfc_albedo, c->ncol * sizeof(float), cudaMemcpyDefault, st));
  else
    RT_CUDA(c, cudaMemcpy2DAsync(albedo, c->ncol * sizeof(float), sfc_albedo, albedo_stride * sizeof(float),
                                 c->ncol * sizeof(float), (size_t)n, cudaMemcpyDefault, st));
  RT_CUDA(c, cudaMemsetAsync(c->bad + first, 0, (size_t)n * sizeof(int), st));
  const unsigned gx = (unsigned)std::min<size_t>((nblk + 255) / 256, (size_t)c->sm_count * 2);
  rt::point_blocks_kernel<<<dim3(gx, (unsigned)n), 256, 0, st>>>(c->blk_max, c->blk_min, tab, c->gas_sum + (size_t)first * nz,
                                                                 c->blk_tab + (size_t)first * nblk, c->ncx / c->mx,
                                                                 c->ncy / c->my, c->ncz / c->mz, c->mz, c->nz,
                                                                 c->merge_ratio, c->bad + first);
  const unsigned ga = (unsigned)std::min<size_t>((c->ncol + 255) / 256, (size_t)c->sm_count * 2);
  rt::albedo_points_kernel<<<dim3(ga, (unsigned)n), 256, 0, st>>>(albedo, c->ncol, broadcast ? 1 : 0, c->bad + first);
  c->launches += 2;
  RT_CUDA(c, cudaGetLastError());
  for (int p = 0; p < n; ++p) c->slot_ok[(size_t)(first + p)] = 2;
  return mark(c, st);
}

int rt_set_points(rt_ctx* c, int first_slot, int n_points, const float* k_abs, const float* k_ray,
                  const float* cloud_ssa, const float* cloud_g, const float* sfc_albedo, uint64_t albedo_stride,
                  void* cuda_stream) {
  if (!c) return RT_EINVAL;
  if (first_slot < 0 || n_points < 1 || first_slot + n_points > c->n_slots)
    return fail(c, RT_EINVAL, "rt_set_points: slots out of range (rt_set_slots)");
  if (!k_abs || !k_ray || !cloud_ssa || !cloud_g || !sfc_albedo) return fail(c, RT_EINVAL, "rt_set_points: NULL argument");
  if (albedo_stride != 0 && albedo_stride < c->ncol) return fail(c, RT_EINVAL, "rt_set_points: albedo_stride must be 0 (one albedo for all points) or >= ncol");
  if (!c->batch_tab) return fail(c, RT_ESTATE, "rt_set_points: call rt_set_slots first");
  if (!c->cloud_ok) return fail(c, RT_ESTATE, "rt_set_points: call rt_set_cloud first");
  for (int p = 0; p < n_points; ++p)
    if (!(cloud_ssa[p] >= 0.0f && cloud_ssa[p] <= 1.0f) || !(std::fabs(cloud_g[p]) < 1.0f))
      return fail(c, RT_EOPTICS, "rt_set_points: cloud_ssa must be in [0, 1] and |cloud_g| < 1");
  if (!fly_mode(c)) {                      // cells of several voxels: a majorant table per point, point by point
    for (int p = 0; p < n_points; ++p)
      if (int rcp = rt_set_point(c, first_slot + p, k_abs + (size_t)p * c->nz, k_ray + (size_t)p * c->nz, cloud_ssa[p],
                                 cloud_g[p], sfc_albedo + (size_t)p * albedo_stride, cuda_stream))
        return rcp;
    return RT_OK;
  }
  DeviceGuard guard(c->device);
  for (int p = 0; p < n_points; ++p) c->slot_ok[(size_t)(first_slot + p)] = 0;
  if (first_slot == 0) c->have_optics = false;
  if (!c->gas_tab) RT_CUDA(c, cudaMalloc(&c->gas_tab, (size_t)c->n_slots * 2 * c->nz * sizeof(float)));
  if (!c->point_par) RT_CUDA(c, cudaMalloc(&c->point_par, (size_t)c->n_slots * sizeof(float2)));
  return set_points_fly(c, first_slot, n_points, k_abs, k_ray, cloud_ssa, cloud_g, sfc_albedo, albedo_stride,
                        (cudaStream_t)cuda_stream);
}

int rt_set_point(rt_ctx* c, int slot, const float* k_abs, const float* k_ray, float cloud_ssa, float cloud_g,
                 const float* sfc_albedo, void* cuda_stream) {
  if (!c) return RT_EINVAL;
  if (slot < 0 || slot >= c->n_slots) return fail(c, RT_EINVAL, "rt_set_point: slot out of range (rt_set_slots)");
  if (!k_abs || !k_ray || !sfc_albedo) return fail(c, RT_EINVAL, "rt_set_point: NULL argument");
  if (!c->batch_tab) return fail(c, RT_ESTATE, "rt_set_point: call rt_set_slots first");
  if (!c->cloud_ok) return fail(c, RT_ESTATE, "rt_set_point: call rt_set_cloud first");
  if (!(cloud_ssa >= 0.0f && cloud_ssa <= 1.0f) || !(std::fabs(cloud_g) < 1.0f))
    return fail(c, RT_EOPTICS, "rt_set_point: cloud_ssa must be in [0, 1] and |cloud_g| < 1");
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  c->slot_ok[slot] = 0;
  if (slot == 0) c->have_optics = false;  // slot 0's majorant and albedo no longer belong to rt_set_optics' packed record
  if (!c->gas_tab) RT_CUDA(c, cudaMalloc(&c->gas_tab, (size_t)c->n_slots * 2 * c->nz * sizeof(float)));
  if (!c->point_par) RT_CUDA(c, cudaMalloc(&c->point_par, (size_t)c->n_slots * sizeof(float2)));
  if (fly_mode(c)) return set_points_fly(c, slot, 1, k_abs, k_ray, &cloud_ssa, &cloud_g, sfc_albedo, 0, st);
  float* tab = c->gas_tab + (size_t)slot * 2 * c->nz;
  const float2 pp = make_float2(cloud_ssa, cloud_g);
  RT_CUDA(c, cudaMemcpyAsync(tab, k_abs, c->nz * sizeof(float), cudaMemcpyDefault, st));
  RT_CUDA(c, cudaMemcpyAsync(tab + c->nz, k_ray, c->nz * sizeof(float), cudaMemcpyDefault, st));
  RT_CUDA(c, cudaMemcpyAsync(c->point_par + slot, &pp, sizeof pp, cudaMemcpyHostToDevice, st));   // pageable: staged before return
  float* albedo = c->albedo + (size_t)slot * c->ncol;
  RT_CUDA(c, cudaMemcpyAsync(albedo, sfc_albedo, c->ncol * sizeof(float), cudaMemcpyDefault, st));
  RT_CUDA(c, cudaMemsetAsync(c->bad + slot, 0, sizeof(int), st));
  if (int rce = ensure_khat_slots(c, slot)) return rce;
  float* khat = c->khat + (size_t)slot * c->ncell;
  const bool merging = c->mx * c->my * c->mz > 1;
  if (merging && !c->kmin) RT_CUDA(c, cudaMalloc(&c->kmin, c->ncell * sizeof(float)));
  rt::point_majorant_kernel<<<c->sm_count * 8, 256, 0, st>>>(c->cloud_max, c->cloud_min, tab, tab + c->nz, khat,
                                                             merging ? c->kmin : nullptr, c->ncx, c->ncy, c->ncz, c->bz, c->bad + slot);
  rt::check_albedo_kernel<<<c->sm_count, 256, 0, st>>>(albedo, c->ncol, c->bad + slot);
  c->launches += 2;
  if (merging) {
    const size_t nblk = c->ncell / ((size_t)c->mx * c->my * c->mz);
    rt::merge_cells_kernel<<<(unsigned)((nblk * 32 + 127) / 128), 128, 0, st>>>(khat, c->kmin, c->ncx, c->ncy, c->ncz,
                                                                                 c->mx, c->my, c->mz, c->merge_ratio);
    ++c->launches;
  }
  RT_CUDA(c, cudaGetLastError());
  c->slot_ok[slot] = 2;
  return mark(c, st);
}

int rt_trace_batch(rt_ctx* c, double zenith_deg, double azimuth_deg, int first_point, int n_points,
                   const uint64_t* counts, uint64_t first_photon_id, uint64_t seed, void* cuda_stream,
                   uint32_t* records_out) {
  if (!c) return RT_EINVAL;
  if (!c->batch_tab) return fail(c, RT_ESTATE, "rt_trace_batch: call rt_set_slots first");
  if (first_point < 0 || n_points < 1 || first_point + n_points > c->n_slots || !counts)
    return fail(c, RT_EINVAL, "rt_trace_batch: points must lie within the slots (rt_set_slots), counts not NULL");
  const char kind = c->slot_ok[first_point];
  for (int j = first_point; j < first_point + n_points; ++j)
    if (c->slot_ok[j] != kind)
      return fail(c, RT_ESTATE, "rt_trace_batch: the points of a launch must all be packed slots or all rt_set_point slots");
  for (int j = first_point; j < first_point + n_points; ++j)
    if (!c->slot_ok[j]) return fail(c, RT_ESTATE, "rt_trace_batch: a slot below n_points has no optics (rt_set_optics_slot)");
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // range errors of the fields of the slots this launch reads (one mask word per slot, cleared when a slot is set again)
  std::vector<int> bad((size_t)n_points, 0);
  RT_CUDA(c, cudaMemcpyAsync(bad.data(), c->bad + first_point, (size_t)n_points * sizeof(int), cudaMemcpyDeviceToHost, st));
  RT_CUDA(c, cudaStreamSynchronize(st));
  for (int j = 0; j < n_points; ++j)
    if (bad[(size_t)j]) {
      char msg[192];
      snprintf(msg, sizeof msg, "rt_trace_batch: slot %d holds input out of range (mask 0x%x: 1 k_ext, 2 k_ext_cloud, 4 ssa, 8 g, 16 albedo)",
               first_point + j, bad[(size_t)j]);
      return fail(c, RT_EOPTICS, msg);
    }
  std::vector<unsigned long long> tab(2 * (size_t)c->n_slots + 1, 0ull);
  unsigned long long total = 0;
  for (int j = 0; j < n_points; ++j) {
    tab[j] = total;
    tab[(size_t)c->n_slots + 1 + j] = (counts[j] / c->ncol) * c->ncol;
    total += counts[j];
  }
  for (int j = n_points; j <= c->n_slots; ++j) tab[j] = total;
  unsigned long long* dtab = c->batch_tab + (c->batch_calls++ & 1u) * tab.size();   // alternate: two launches in flight
  RT_CUDA(c, cudaMemcpyAsync(dtab, tab.data(), tab.size() * sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
  RT_CUDA(c, cudaStreamSynchronize(st));   // tab is a stack vector
  return do_trace(c, zenith_deg, azimuth_deg, total, first_photon_id, seed, 0u, cuda_stream, records_out, n_points,
                  first_point, dtab, kind == 2);
}

int rt_trace(rt_ctx* c, double zenith_deg, double azimuth_deg, uint64_t n_photons, uint64_t first_photon_id,
             uint64_t seed, uint32_t stream_id, void* cuda_stream) {
  return do_trace(c, zenith_deg, azimuth_deg, n_photons, first_photon_id, seed, stream_id, cuda_stream, nullptr);
}

int rt_trace_range(rt_ctx* c, double zenith_deg, double azimuth_deg, uint64_t job_photons, uint64_t first_photon_id,
                   uint64_t seed, uint32_t stream_id, void* cuda_stream, uint64_t range_begin, uint64_t range_count,
                   uint32_t* records_out) {
  if (c && (range_begin > job_photons || range_count > job_photons - range_begin))
    return fail(c, RT_EINVAL, "rt_trace_range: the range must lie within [0, job_photons)");
  return do_trace(c, zenith_deg, azimuth_deg, range_count, first_photon_id, seed, stream_id, cuda_stream, records_out,
                  0, 0, nullptr, false, range_begin, job_photons);
}

int rt_trace_records(rt_ctx* c, double zenith_deg, double azimuth_deg, uint64_t n_photons,
                     uint64_t first_photon_id, uint64_t seed, uint32_t stream_id, void* cuda_stream,
                     uint32_t* records_out) {
  if (c && !records_out && n_photons) return fail(c, RT_EINVAL, "rt_trace_records: NULL records_out");
  return do_trace(c, zenith_deg, azimuth_deg, n_photons, first_photon_id, seed, stream_id, cuda_stream, records_out);
}

int rt_read_tallies(rt_ctx* c, int64_t* atm_abs, int64_t* sfc_dir, int64_t* sfc_dif, int64_t* sfc_abs,
                    int64_t* toa_up, rt_counters* counters) {
  if (!c) return RT_EINVAL;
  DeviceGuard guard(c->device);
  if (int rcw = wait_pending(c)) return rcw;   // this context's work only, not the whole device
  int64_t* outs[5] = {atm_abs, sfc_dir, sfc_dif, sfc_abs, toa_up};
  for (int k = 0; k < 5; ++k)
    if (outs[k])
      RT_CUDA(c, cudaMemcpyAsync(outs[k], tally_ptr(c, k), (k == 0 ? c->nvox : c->ncol) * sizeof(int64_t), cudaMemcpyDefault, c->copy_stream));
  unsigned long long h[rt::C_COUNT];
  if (counters) RT_CUDA(c, cudaMemcpyAsync(h, c->counters, sizeof h, cudaMemcpyDeviceToHost, c->copy_stream));
  RT_CUDA(c, cudaStreamSynchronize(c->copy_stream));
  if (counters) fill_counters(h, counters);
  return RT_OK;
}

int rt_read_tallies_async(rt_ctx* c, int64_t* atm_abs, int64_t* sfc_dir, int64_t* sfc_dif, int64_t* sfc_abs,
                          int64_t* toa_up, rt_counters* counters, void* cuda_stream) {
  if (!c) return RT_EINVAL;
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int64_t* outs[5] = {atm_abs, sfc_dir, sfc_dif, sfc_abs, toa_up};
  for (int k = 0; k < 5; ++k)
    if (outs[k])
      RT_CUDA(c, cudaMemcpyAsync(outs[k], tally_ptr(c, k), (k == 0 ? c->nvox : c->ncol) * sizeof(int64_t), cudaMemcpyDefault, st));
  if (counters) {
    // No kernel here: behind a persistent trace kernel of ANOTHER context that already fills the SMs (it starts in the
    // tail of this context's trace), a kernel of this stream would wait for that whole trace, and with it the caller's
    // wait for this read-out and the upload of its next step (5.5 ms per step in bench.py's e2e leg).
    if (!c->counter_jobs) RT_CUDA(c, cudaHostAlloc(&c->counter_jobs, 2 * sizeof(rt_ctx::CounterJob), cudaHostAllocDefault));
    rt_ctx::CounterJob* job = c->counter_jobs + (c->counter_calls++ & 1u);
    job->out = counters;
    RT_CUDA(c, cudaMemcpyAsync(job->raw, c->counters, sizeof job->raw, cudaMemcpyDeviceToHost, st));
    RT_CUDA(c, cudaLaunchHostFunc(st, counters_host_fn, job));
  }
  RT_CUDA(c, cudaGetLastError());
  return mark(c, st);
}

int rt_set_merge(rt_ctx* c, int mx, int my, int mz, float merge_ratio) {
  if (!c) return RT_EINVAL;
  auto pow2 = [](int v) { return v > 0 && !(v & (v - 1)); };
  if (!pow2(mx) || !pow2(my) || !pow2(mz) || c->ncx % mx || c->ncy % my || c->ncz % mz || mx > 64 || my > 64 || mz > 64)
    return fail(c, RT_EINVAL, "rt_set_merge: factors must be powers of two <= 64 dividing the acceleration grid");
  if (!(merge_ratio >= 1.0f) || !std::isfinite(merge_ratio)) return fail(c, RT_EINVAL, "rt_set_merge: merge_ratio must be >= 1");
  c->mx = mx; c->my = my; c->mz = mz; c->merge_ratio = merge_ratio;
  c->have_optics = false;                 // every majorant table was built for the old factors: all slots
  for (auto& ok : c->slot_ok) ok = 0;     // must be given optics again (RT_ESTATE otherwise)
  c->cloud_ok = false;                    // ... and the cloud field's block tables (rt_set_cloud) too
  if (c->blk_tab) {
    DeviceGuard guard(c->device);
    if (int rcw = wait_pending(c)) return rcw;
    cudaFree(c->blk_tab); c->blk_tab = nullptr;
  }
  return RT_OK;
}

int rt_set_source(rt_ctx* c, float diffuse_fraction, int sampler) {
  if (!c) return RT_EINVAL;
  if (!(diffuse_fraction >= 0.0f && diffuse_fraction <= 1.0f)) return fail(c, RT_EINVAL, "rt_set_source: diffuse_fraction must be in [0, 1]");
  if (sampler != RT_SAMPLER_PHILOX && sampler != RT_SAMPLER_SOBOL) return fail(c, RT_EINVAL, "rt_set_source: unknown sampler");
  c->diffuse_fraction = diffuse_fraction; c->sobol = (sampler == RT_SAMPLER_SOBOL);
  return RT_OK;
}

int rt_set_heating_split(rt_ctx* c, int on) {
  if (!c) return RT_EINVAL;
  DeviceGuard guard(c->device);
  if (on && !c->atm_dir) {
    RT_CUDA(c, cudaMalloc(&c->atm_dir, c->nvox * sizeof(unsigned long long)));
    RT_CUDA(c, cudaMemset(c->atm_dir, 0, c->nvox * sizeof(unsigned long long)));
  }
  c->split = on != 0;
  return RT_OK;
}

int rt_read_heating_direct(rt_ctx* c, int64_t* out) {
  if (!c || !out) return RT_EINVAL;
  if (!c->atm_dir) return fail(c, RT_ESTATE, "rt_read_heating_direct: call rt_set_heating_split(ctx, 1) first");
  DeviceGuard guard(c->device);
  if (int rcw = wait_pending(c)) return rcw;
  RT_CUDA(c, cudaMemcpyAsync(out, c->atm_dir, c->nvox * sizeof(int64_t), cudaMemcpyDefault, c->copy_stream));
  RT_CUDA(c, cudaStreamSynchronize(c->copy_stream));
  return RT_OK;
}

int rt_set_mode(rt_ctx* c, int mode) {
  if (!c) return RT_EINVAL;
  if (mode != RT_MODE_ANALOG && mode != RT_MODE_WEIGHTED) return fail(c, RT_EINVAL, "rt_set_mode: unknown mode");
  c->weighted = (mode == RT_MODE_WEIGHTED);
  return RT_OK;
}

int rt_tally_to_flux(const int64_t* tally, double* out, uint64_t count, uint64_t n_photons, uint64_t ncol,
                     double tod_flux, double depth) {
  if (!tally || !out || n_photons == 0 || ncol == 0) return RT_EINVAL;
  if (!(tod_flux >= 0.0) || !std::isfinite(tod_flux) || !(depth >= 0.0) || !std::isfinite(depth)) return RT_EINVAL;
  const double per_quantum = tod_flux * (double)ncol / (double)n_photons / (double)RT_W0 / (depth > 0.0 ? depth : 1.0);
  for (uint64_t k = 0; k < count; ++k) out[k] = (double)tally[k] * per_quantum;
  return RT_OK;
}

int rt_reset_tallies(rt_ctx* c, void* cuda_stream) {
  if (!c) return RT_EINVAL;
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  RT_CUDA(c, cudaMemsetAsync(c->tallies, 0, (c->nvox + 4 * c->ncol) * sizeof(unsigned long long), st));
  RT_CUDA(c, cudaMemsetAsync(c->counters, 0, (rt::C_COUNT + 1) * sizeof(unsigned long long), st));
  if (c->atm_dir) RT_CUDA(c, cudaMemsetAsync(c->atm_dir, 0, c->nvox * sizeof(unsigned long long), st));
  return mark(c, st);
}

int rt_read_majorant(rt_ctx* c, float* khat_out) {
  if (!c || !khat_out) return RT_EINVAL;
  if (c->slot_ok[0] == 2 && fly_mode(c))
    return fail(c, RT_ESTATE, "rt_read_majorant: rt_set_point keeps no majorant table for voxel-sized merged cells");
  DeviceGuard guard(c->device);
  if (int rcw = wait_pending(c)) return rcw;
  RT_CUDA(c, cudaMemcpyAsync(khat_out, c->khat, c->ncell * sizeof(float), cudaMemcpyDefault, c->copy_stream));
  RT_CUDA(c, cudaStreamSynchronize(c->copy_stream));
  return RT_OK;
}

int rt_read_packed_optics(rt_ctx* c, float* packed_out) {
  if (!c || !packed_out) return RT_EINVAL;
  DeviceGuard guard(c->device);
  if (int rcw = wait_pending(c)) return rcw;
  RT_CUDA(c, cudaMemcpyAsync(packed_out, c->optics, c->nvox * sizeof(float4), cudaMemcpyDefault, c->copy_stream));
  RT_CUDA(c, cudaStreamSynchronize(c->copy_stream));
  return RT_OK;
}

int rt_gather_bench(rt_ctx* c, uint32_t loads_per_thread, uint64_t footprint_voxels, void* cuda_stream,
                    float* ms_out, uint64_t* n_loads_out) {
  if (!c || !ms_out || !n_loads_out || loads_per_thread < 8 || footprint_voxels > c->nvox) return RT_EINVAL;
  const unsigned long long nfoot = footprint_voxels ? footprint_voxels : c->nvox;
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const uint32_t iters = loads_per_thread / 8;
  const int blocks = c->sm_count * 8, threads = 256;
  cudaEvent_t a, b;
  RT_CUDA(c, cudaEventCreate(&a));
  RT_CUDA(c, cudaEventCreate(&b));
  rt::gather_bench_kernel<<<blocks, threads, 0, st>>>(c->optics, nfoot, iters, c->sink);   // warm-up
  RT_CUDA(c, cudaEventRecord(a, st));
  rt::gather_bench_kernel<<<blocks, threads, 0, st>>>(c->optics, nfoot, iters, c->sink);
  c->launches += 2;
  RT_CUDA(c, cudaEventRecord(b, st));
  RT_CUDA(c, cudaEventSynchronize(b));
  RT_CUDA(c, cudaGetLastError());
  RT_CUDA(c, cudaEventElapsedTime(ms_out, a, b));
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  *n_loads_out = (uint64_t)blocks * threads * iters * 8ull;
  return RT_OK;
}

int rt_last_trace_ms(rt_ctx* c, float* ms_out) {
  if (!c || !ms_out) return RT_EINVAL;
  if (!c->have_trace) return fail(c, RT_ESTATE, "rt_last_trace_ms: no rt_trace call yet");
  DeviceGuard guard(c->device);
  RT_CUDA(c, cudaEventSynchronize(c->ev1));
  RT_CUDA(c, cudaEventElapsedTime(ms_out, c->ev0, c->ev1));
  return RT_OK;
}

uint64_t rt_launch_count(const rt_ctx* c) { return c ? c->launches : 0; }

int rt_philox_words(int cuda_device, const uint32_t* ctr, uint32_t key0, uint32_t key1, uint32_t* out, uint64_t n) {
  if (!ctr || !out) return RT_EINVAL;
  DeviceGuard guard(cuda_device);
  if (n == 0) return RT_OK;
  rt::philox_words_kernel<<<296, 256>>>((const uint4*)ctr, key0, key1, (uint4*)out, n);
  if (cudaGetLastError() != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) return RT_ECUDA;
  return RT_OK;
}

int rt_selftest_ieee(int cuda_device, uint64_t* rcp_mismatches, uint64_t* sqrt_mismatches) {
  if (!rcp_mismatches || !sqrt_mismatches) return RT_EINVAL;
  DeviceGuard guard(cuda_device);
  unsigned long long* d = nullptr;
  if (cudaMalloc(&d, 2 * sizeof(unsigned long long)) != cudaSuccess) return RT_ENOMEM;
  unsigned long long h[2] = {0, 0};
  cudaError_t ce = cudaMemset(d, 0, sizeof h);
  // reciprocal: biased exponents 1 .. 251 (2^-126 <= |x| < 2^125); square root: from 2^-101 to the largest finite float
  if (ce == cudaSuccess) {
    rt::ieee_selftest_kernel<<<1184, 256>>>(d, 1u << 23, 252u << 23, 0x0d000000u, 0x7f800000u);
    ce = cudaGetLastError();
  }
  if (ce == cudaSuccess) ce = cudaMemcpy(h, d, sizeof h, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (ce != cudaSuccess) return RT_ECUDA;
  *rcp_mismatches = h[0]; *sqrt_mismatches = h[1];
  return RT_OK;
}

const char* rt_last_error(const rt_ctx* c) { return c ? c->err.c_str() : "null context"; }

void rt_destroy(rt_ctx* c) {
  if (!c) return;
  {
    DeviceGuard guard(c->device);
    cudaDeviceSynchronize();
    cudaFree(c->optics); cudaFree(c->khat); cudaFree(c->kmin); cudaFree(c->atm_dir); cudaFree(c->albedo); cudaFree(c->tallies);
    cudaFree(c->counters); if (c->counter_jobs) cudaFreeHost(c->counter_jobs); cudaFree(c->bad); cudaFree(c->gas_tab); cudaFree(c->point_par);
    cudaFree(c->cloud); cudaFree(c->cloud_max); cudaFree(c->cloud_min); cudaFree(c->batch_tab); cudaFree(c->sink); cudaFree(c->stage);
    cudaFree(c->blk_max); cudaFree(c->blk_min); cudaFree(c->blk_tab); cudaFree(c->gas_sum);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    for (auto& p : c->pending) cudaEventDestroy(p.second);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  }
  delete c;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------------------------
// rt_majorant_no_alloc (include/rt.h): the majorant table of §3.5 + §3.5b for callers that must not allocate.
// The scratch of the step (the per-cell minima of the merge criterion, which rt_set_optics keeps in a cudaMalloc'ed
// array of the context) is this file-scope device array.  Device code names it directly; HOST code must not pass the
// name to a kernel (on the host it is a stand-in, not a device address): the address is asked for once per device
// with cudaGetSymbolAddress, below.
static __device__ __align__(256) float g_no_alloc_cell_min[RT_NO_ALLOC_MAX_CELLS];

namespace {

// Variant of the cell-extrema step of the pack kernels for the extinction field alone: one thread per acceleration
// cell; the cell's maximum goes to the caller's table, its minimum to the scratch array (every cell the merge step
// reads is written here first, so what an earlier call left in the array never matters).
__global__ void cell_extrema_no_alloc_kernel(const float* __restrict__ k_ext, float* __restrict__ khat, int nx, int ny,
                                             int nz, int bx, int by, int bz, int* __restrict__ bad) {
  const int ncx = nx / bx, ncy = ny / by, ncz = nz / bz;
  const size_t ncell = (size_t)ncx * ncy * ncz;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  bool ok = true;
  for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < ncell; c += stride) {
    const int cx = (int)(c % ncx), cy = (int)((c / ncx) % ncy), cz = (int)(c / ((size_t)ncx * ncy));
    float hi = 0.0f, lo = INFINITY;
    for (int z = cz * bz; z < (cz + 1) * bz; ++z)
      for (int y = cy * by; y < (cy + 1) * by; ++y)
        for (int x = cx * bx; x < (cx + 1) * bx; ++x) {
          const float k = __ldg(k_ext + ((size_t)z * ny + y) * nx + x);
          if (!(k >= 0.0f) || isinf(k)) ok = false;
          hi = fmaxf(hi, k); lo = fminf(lo, k);
        }
    khat[c] = hi;
    g_no_alloc_cell_min[c] = lo;
  }
  if (!ok && bad) atomicOr(bad, 1);
}

constexpr int kNoAllocMaxDevices = 64;
float* g_no_alloc_ptr[kNoAllocMaxDevices] = {};   // device address of g_no_alloc_cell_min per device, once known
int g_no_alloc_sms[kNoAllocMaxDevices] = {};
std::mutex g_no_alloc_mutex;
thread_local char g_no_alloc_err[256] = "";

int no_alloc_fail(int code, const char* fmt, unsigned long long a = 0, unsigned long long b = 0) {
  snprintf(g_no_alloc_err, sizeof g_no_alloc_err, fmt, a, b);
  return code;
}

}  // namespace

extern "C" {

const char* rt_no_alloc_last_error(void) { return g_no_alloc_err; }

int rt_majorant_no_alloc(const float* k_ext, float* khat_out, int* bad_out, int nx, int ny, int nz, int bx, int by,
                         int bz, int mx, int my, int mz, float merge_ratio, int cuda_device, void* cuda_stream) {
  if (!k_ext || !khat_out) return no_alloc_fail(RT_EINVAL, "rt_majorant_no_alloc: NULL field or table");
  if (nx <= 0 || ny <= 0 || nz <= 0 || bx <= 0 || by <= 0 || bz <= 0 || nx % bx || ny % by || nz % bz)
    return no_alloc_fail(RT_EINVAL, "rt_majorant_no_alloc: sizes must be positive and the block must divide the grid");
  const int ncx = nx / bx, ncy = ny / by, ncz = nz / bz;
  const unsigned long long ncell = (unsigned long long)ncx * ncy * ncz;
  if (ncell > (unsigned long long)RT_NO_ALLOC_MAX_CELLS)
    return no_alloc_fail(RT_EINVAL, "rt_majorant_no_alloc: %llu acceleration cells exceed RT_NO_ALLOC_MAX_CELLS = %llu "
                         "(the scratch array is fixed; use rt_set_optics on a context)", ncell, RT_NO_ALLOC_MAX_CELLS);
  auto pow2 = [](int v) { return v > 0 && !(v & (v - 1)); };
  if (!pow2(mx) || !pow2(my) || !pow2(mz) || ncx % mx || ncy % my || ncz % mz || mx > 64 || my > 64 || mz > 64)
    return no_alloc_fail(RT_EINVAL, "rt_majorant_no_alloc: merge factors must be powers of two <= 64 dividing the acceleration grid");
  if (!(merge_ratio >= 1.0f) || !std::isfinite(merge_ratio))
    return no_alloc_fail(RT_EINVAL, "rt_majorant_no_alloc: merge_ratio must be >= 1");
  if (cuda_device < 0 || cuda_device >= kNoAllocMaxDevices)
    return no_alloc_fail(RT_EINVAL, "rt_majorant_no_alloc: device %llu out of range", (unsigned long long)cuda_device);
  DeviceGuard guard(cuda_device);
  float* scratch = nullptr;
  int sms = 0;
  {
    // set-up, once per device, with that device current: the DEVICE address of the scratch array
    std::lock_guard<std::mutex> lock(g_no_alloc_mutex);
    if (!g_no_alloc_ptr[cuda_device]) {
      float* p = nullptr;
      cudaError_t ce = cudaGetSymbolAddress((void**)&p, g_no_alloc_cell_min);
      if (ce != cudaSuccess || !p) {
        snprintf(g_no_alloc_err, sizeof g_no_alloc_err, "rt_majorant_no_alloc: cudaGetSymbolAddress: %s", cudaGetErrorString(ce));
        return RT_ECUDA;
      }
      int n = 0;
      ce = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, cuda_device);
      if (ce != cudaSuccess || n < 1) {
        snprintf(g_no_alloc_err, sizeof g_no_alloc_err, "rt_majorant_no_alloc: cudaDeviceGetAttribute: %s", cudaGetErrorString(ce));
        return RT_ECUDA;
      }
      g_no_alloc_sms[cuda_device] = n;
      g_no_alloc_ptr[cuda_device] = p;
    }
    scratch = g_no_alloc_ptr[cuda_device];
    sms = g_no_alloc_sms[cuda_device];
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaError_t ce = cudaSuccess;
  if (bad_out) ce = cudaMemsetAsync(bad_out, 0, sizeof(int), st);
  if (ce == cudaSuccess) {
    const unsigned blocks = (unsigned)std::min<unsigned long long>((ncell + 255) / 256, (unsigned long long)sms * 8);
    cell_extrema_no_alloc_kernel<<<blocks, 256, 0, st>>>(k_ext, khat_out, nx, ny, nz, bx, by, bz, bad_out);
    if (mx * my * mz > 1) {
      const unsigned long long nblk = ncell / ((unsigned long long)mx * my * mz);
      rt::merge_cells_kernel<<<(unsigned)((nblk * 32 + 127) / 128), 128, 0, st>>>(khat_out, scratch, ncx, ncy, ncz, mx, my,
                                                                                   mz, merge_ratio);
    }
    ce = cudaGetLastError();
  }
  if (ce != cudaSuccess) {
    snprintf(g_no_alloc_err, sizeof g_no_alloc_err, "rt_majorant_no_alloc: %s", cudaGetErrorString(ce));
    return RT_ECUDA;
  }
  return RT_OK;
}

}  // extern "C"
