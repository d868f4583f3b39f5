// rt_trace.cuh — the persistent photon-tracing kernel.
//
// One thread carries one photon at a time.  Its position inside the current acceleration cell is held
// as the remaining distances (rx, ry, rz) along the flight direction to the cell's next face on each
// axis: a cell crossing is ~25 arithmetic instructions (smallest of three, two subtractions, one
// reset to the face spacing, index step) and one 4-byte load of the majorant.  With crossings that cheap the
// acceleration grid can be as fine as the simulation grid where the medium is not homogeneous: cells of ONE voxel
// (merged 8^3 where the air is clear) have the voxel's own extinction as majorant, so there are no
// null collisions outside merged cells: 15.8 tentative collisions and 77 crossings per photon on the 512x512x128
// cumulus field, against 38 + 58 with 2^3-voxel cells and 202 + 42 with 8^3.
//
// Divergence.  The cheap step, MOVE (find the nearest face; cross it, change level if the entered cell is at the
// other level, or notice that the tentative collision comes first), is what live lanes do by default, in a ROLLED
// loop (one copy: the kernel is larger than the instruction cache and reacts to every added copy).  The expensive
// steps are each wanted by few lanes per iteration -- a collision (voxel gather, classification, Philox draw,
// logarithm), a real scatter (phase-function inversion, rotation, three reciprocals), a surface or domain-top
// arrival -- and run inline they executed with 2-6 lanes active.  So a lane that needs one PARKS in COLLIDE, SCATTER
// or BOUNDARY, and the warp votes to run that phase once enough lanes wait for it; DEAD lanes are refilled
// kRegenBatch at a time from a warp-private pool of photon ids taken in chunks from a global counter
// (BASELINE.json north_star: "compacted and regenerated persistently with warp-level ballot/shuffle").  A photon's own
// sequence of arithmetic operations does not depend on the scheduling, so neither do the results.
#pragma once
#include "rt_device.cuh"

namespace rt {

constexpr unsigned long long kW0 = 1ull << 32;  // tally quanta per photon
constexpr uint32_t kEventCap = 1u << 20;        // §3.12
constexpr float kTiny = 1e-30f;                 // direction components are nudged away from 0
constexpr int kTraceThreads = 256;
constexpr int kChunk = 128;                     // photon ids a warp takes per global atomic (fewer in small launches)
// Vote thresholds: a parked phase runs when this many lanes wait for it (or nothing can move).  COLLIDE's threshold and
// the MOVE steps between two votes depend on the acceleration grid (TraceArgs::vote_bias, move_steps, set by rt.cu):
// with voxel-sized cells a photon crosses ~5 cells per collision instead of ~1.5, so batches take longer to fill
// (sweeps: profiles/r1_block_sweep.md, r2_pool_kernel.md, r2_trace_kernel.md).
constexpr int kMinBlocks = 4;          // resident blocks per SM the launch bounds ask for (64 registers)
constexpr int kRegenBatch = 6;         // refill when this many lanes are idle (or nothing else to do)
constexpr int kScatterBatch = 8;       // SCATTER
constexpr int kCollideBatch = 8, kCollideBatchUnit = 12;   // COLLIDE: cells of several voxels / voxel-sized cells
constexpr int kBoundaryBatch = 8;      // BOUNDARY: surface and domain-top arrivals (1 per photon)
constexpr int kMoveSteps = 3, kMoveStepsUnit = 5;           // MOVE steps between two votes
constexpr int kMoveStepsFly = 6;       // ... in a sweep over spectral points kept factored (8 crossings per collision)
constexpr unsigned vote_bias(int collide_batch) {
  return (32u - kRegenBatch) | ((32u - 1u) << 6) | ((32u - (unsigned)collide_batch) << 12) |
         ((32u - kScatterBatch) << 18) | ((32u - kBoundaryBatch) << 24);
}

enum Counter { C_NULL = 0, C_RAY, C_HG, C_ATM_ABS, C_SFC_HITS, C_SFC_ABS, C_TOA, C_CAPPED, C_CELLS,
               C_CAPPED_E, C_RELEVEL, C_ROUL_KILLED, C_ROUL_KEPT, C_ROUL_LOST, C_ROUL_GAINED, C_COUNT };

enum : uint32_t { ST_DEAD = 0, ST_MOVE = 1, ST_COLLIDE = 2, ST_SCATTER = 3, ST_BOUNDARY = 4 };

struct TraceArgs {
  int nx, ny, nz, bx, by, bz, ncx, ncy, ncz;
  float dx, dy, dz, rdx, rdy, rdz, Lx, Ly, Lz;
  float rLx, rLy, rLz;                 // 1 / Lx ...: §3.7b counts the whole cells in a remaining distance without dividing
  // §3.5b merged cells: factors (powers of two), their reciprocals, merged-cell extents (m b) d
  int mx, my, mz;
  float rmx, rmy, rmz, Lx1, Ly1, Lz1;
  unsigned vote_bias;                  // thresholds of the vote (vote_bias() above)
  // kPow2: the cell index (cx, cy, cz) lives in ONE word, pc = cz << shz | cy << lx | cx, which for power-of-two ncx,
  // ncy is the linear index of the cell in the majorant table; a crossing is one add and one masked merge, the
  // periodic wrap is the field mask.  zmask = the bits from shz up; omask clears the in-block bits of the three
  // fields (origin of a merged cell).  rt.cu uses these instantiations only when ncell + 64 ncx ncy < 2^31, so that
  // a step beyond the top stays positive as an int and a step below the surface is negative.
  int lx, shz;
  unsigned xmask, ymask, zmask, omask;
  int move_steps;                      // MOVE steps between two votes: kMoveSteps or kMoveStepsUnit
  int unit;                            // bx = by = bz = 1: a level-0 acceleration cell IS a voxel (no position needed to
                                       // find the collision's voxel, and no null collisions outside merged cells)
  float sun_x, sun_y, sun_z, sun_ix, sun_iy, sun_iz;  // beam direction and 1/nudge(component), host-computed
  const float4* __restrict__ optics;   // [z][y][x] (c1, c2, c3, g)
  const float* __restrict__ khat;      // [cz][cy][cx]
  const float* __restrict__ albedo;    // [y][x]
  unsigned long long* atm_abs;         // [z][y][x]
  unsigned long long* atm_dir;         // [z][y][x] or nullptr: the part of atm_abs from never-scattered photons
  unsigned long long *sfc_dir, *sfc_dif, *sfc_abs, *toa_up;  // [y][x]
  unsigned long long* counters;        // C_COUNT words
  unsigned long long* next_photon;     // work counter, zeroed before launch
  uint32_t* records;                   // 4 words per photon or nullptr
  unsigned long long n_photons, first_id, n_full, ncol;   // photons of this launch; id of the JOB's photon 0; job's full passes
  unsigned long long index_base;       // index in the job of this launch's first photon (rt_trace: 0; rt_trace_range: range_begin)
  unsigned chunk;                      // photon ids per global atomic: kChunk, or less so that a small launch still spreads over all warps
  PhiloxKeys keys;                     // round keys of the Philox key (seed)
  PhiloxKeys keys_sobol;               // ... of (seed low, seed high ^ 'SOBL'): digital shifts of §3.15
  // batched launch (kBatch; rt_trace_batch): photons of n_points spectral points in one launch; point j owns
  // the launch indices [offsets[j], offsets[j+1]), reads optics slot j and majorant slot j, draws on stream j
  const unsigned long long* offsets;   // n_points + 1 prefix sums (device)
  const unsigned long long* nfull;     // per point: ncol * floor(count / ncol) (device)
  int n_points, first_point;           // points first_point .. first_point + n_points - 1 (slot = stream id = point)
  unsigned nvox32, ncell32, ncol32;    // slot strides of optics, majorant and albedo
  // factored optics in the trace (kBatch only; rt_set_cloud / rt_set_point): COLLIDE builds the voxel's record from
  // the shared cloud field and the point's tables with the operations of §3.4b + §3.4 instead of gathering it
  const float* cloud;                  // [z][y][x] or nullptr (then the packed slots are used)
  const float* gas;                    // per point: k_abs[nz] then k_ray[nz]
  const float2* point_par;             // per point: (cloud_ssa, cloud_g)
  // ... with voxel-sized cells and merging (fly): no majorant table per point.  A voxel's majorant is its own
  // fl((k_abs[z] + k_ray[z]) + k_cloud), read from the shared cloud field; per point only one word per block of
  // merged cells (sign bit set: merged, |word| = the block's maximum) and the gas sums per level
  int fly;
  const float* btab;                   // [point][block]
  const float* gsum;                   // [point][nz]
  int lmx, lmy, lmz, nbx, nby;         // log2 of the merge factors, blocks per row / column
  unsigned nblk32;                     // slot stride of btab
  float diffuse_fraction;              // §3.15: share of photons launched diffusely (0: none)
  int sobol;                           // §3.15: entry points from the scrambled 2-D Sobol sequence
  uint32_t stream_id;
};

// Add kW0 to *p once per distinct address among the lanes of `mask` (warp-aggregated tally).
__device__ __forceinline__ void tally_add(unsigned mask, unsigned long long* p) {
  const unsigned peers = __match_any_sync(mask, (unsigned long long)p);
  if ((unsigned)(__ffs(peers) - 1) == (threadIdx.x & 31u))
    atomicAdd(p, kW0 * (unsigned long long)__popc(peers));
}

__device__ __forceinline__ float nudge(float d) { return fabsf(d) < kTiny ? kTiny : d; }

__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
  return v;
}



// kPow2: the acceleration grid's x and y extents are powers of two, so the periodic wrap is a mask.
// kWeighted: the paper's absorption weights + Russian roulette instead of analog
// absorption: integer weight wq (tally quanta), deposits at every tentative collision, roulette ledger.
// kBatch: several spectral points in one launch, each with its own optics and majorant slot (see TraceArgs).
template <bool kRecords, bool kPow2, bool kWeighted, bool kBatch = false>
// Launch bounds: 4 blocks of 256 threads per SM (64 registers) for the weighted and the batch instantiations; the
// analog single-point ones need 58 registers and run better squeezed to 48 with 5 blocks per SM (40 warps instead of
// 32 hide more of the majorant load's latency: config 3 67.8 -> 67.2 ms, config 5 379 -> 368; weighted 74.4 -> 75.1 and
// the batch kernel 49.9 -> 50.4 would lose).
__global__ void __launch_bounds__(kTraceThreads, (!kBatch && !kWeighted) ? kMinBlocks + 1 : kMinBlocks) trace_kernel(const TraceArgs A) {
  __shared__ unsigned long long s_cnt[C_COUNT];
  // finished photons of this block per fate (1..5): 32-bit words, because a 64-bit shared-memory atomic is a
  // compare-and-swap loop; a launch holds fewer than 2^32 photons (rt.cu splits longer calls)
  __shared__ unsigned s_fate[8];
  if (threadIdx.x < C_COUNT) s_cnt[threadIdx.x] = 0ull;
  if (threadIdx.x < 8) s_fate[threadIdx.x] = 0u;
  __syncthreads();

  const unsigned lane = threadIdx.x & 31u;
  const unsigned lt_mask = (1u << lane) - 1u;
  unsigned long long pool_next = 0, pool_end = 0;  // warp-uniform chunk of photon indices
  bool exhausted = false;                          // warp-uniform: the global counter has run out

  // photon state
  uint32_t st = ST_DEAD;
  unsigned long long i = 0;               // index in the call (kBatch: in the photon's point)
  uint32_t jpt = 0;                       // kBatch: the photon's point = its stream id and slot
  unsigned long long ig = 0;              // kBatch: index in the launch (records)
  uint32_t e = 0;
  int cx = 0, cy = 0, cz = 0;             // the cell (generic grids)
  uint32_t pc = 0;                        // ... packed (kPow2), see TraceArgs
  uint32_t dpx = 0, dpy = 0, dpz = 0;     // kPow2: the index step per axis (+-1, or +-m in a merged cell) in its field's position
  auto X = [&]() -> int { if constexpr (kPow2) return (int)(pc & A.xmask); else return cx; };
  auto Y = [&]() -> int { if constexpr (kPow2) return (int)((pc & A.ymask) >> A.lx); else return cy; };
  auto Z = [&]() -> int { if constexpr (kPow2) return (int)pc >> A.shz; else return cz; };   // arithmetic: < 0 below the surface
  auto set_cell = [&](int x, int y, int z) {
    if constexpr (kPow2) pc = ((uint32_t)z << A.shz) | ((uint32_t)y << A.lx) | (uint32_t)x;
    else { cx = x; cy = y; cz = z; }
  };
  auto add_x = [&](int v) { if constexpr (kPow2) pc += (uint32_t)v; else cx += v; };          // within a block: no carry
  auto add_y = [&](int v) { if constexpr (kPow2) pc += (uint32_t)v << A.lx; else cy += v; };
  auto add_z = [&](int v) { if constexpr (kPow2) pc += (uint32_t)v << A.shz; else cz += v; };
  float da = 0, db = 0, dc = -1;          // unit direction
  float rx = 0, ry = 0, rz = 0;           // remaining distance to the cell's next face on each axis
  float delx = 0, dely = 0, delz = 0;     // distance between successive faces on each axis
  float tau = 0, kh = 0, u1 = 0;
  uint32_t w2 = 0, w3 = 0;                // words 2, 3 of the current event's draw
  uint32_t sw2 = 0, sw3 = 0;              // ... of the event that chose SCATTER (its draw is already replaced)
  float sg = 0;                           // asymmetry parameter for the pending scatter; 2 = Rayleigh
  bool direct = true;
  // §3.7b: kh holds the majorant table's word as stored, i.e. its sign bit says whether the photon travels
  // through a merged cell (then cx, cy, cz = that cell's origin); the majorant itself is |kh|
  uint32_t stp = 0;                       // generic grids: index step per axis as three signed bytes (+-1, or +-m in a
                                          // merged cell)
  // event counts: running totals of this thread; a photon's own counts are differences (records)
  uint32_t t_ev = 0, t_sc = 0, t_hg = 0, t_sfc = 0, t_cells = 0, t_relevel = 0;
  unsigned long long wq = kW0;            // weighted mode: the photon's weight in tally quanta
  unsigned long long t_rlost = 0, t_rgain = 0;   // roulette ledger of this thread

  uint32_t t_rkept = 0;
  uint32_t b_ev = 0, b_sc = 0, b_sfc = 0;  // totals when the current photon was launched (records only)

  auto sid = [&]() { return kBatch ? jpt : A.stream_id; };
  auto draw = [&]() {
    const unsigned long long pid = A.first_id + A.index_base + i;
    const uint4 X = philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), e, sid(), A.keys);
    tau = neg_log(1.0f - u24(X.x)); u1 = u24(X.y); w2 = X.z; w3 = X.w;
  };
  // local coordinate from a remaining distance: q = face - v r, face = L if v > 0 else 0
  auto local = [&](float v, float r, float L) {   // v: a direction component as set by place(), i.e. nudged (Q20)
    return fminf(L, fmaxf(0.0f, fmaf(-v, r, v > 0.0f ? L : 0.0f)));
  };
  // after a change of direction at local position (qx, qy, qz): reciprocals, face spacings, distances
  auto set_steps = [&](bool lev) {
    const int ax_ = (da > 0.0f) ? 1 : -1, ay_ = (db > 0.0f) ? 1 : -1, az_ = (dc > 0.0f) ? 1 : -1;
    const int sx = lev ? ax_ * A.mx : ax_, sy = lev ? ay_ * A.my : ay_, sz = lev ? az_ * A.mz : az_;
    if constexpr (kPow2) { dpx = (uint32_t)sx; dpy = (uint32_t)sy << A.lx; dpz = (uint32_t)sz << A.shz; }
    else stp = ((uint32_t)sx & 0xffu) | (((uint32_t)sy & 0xffu) << 8) | (((uint32_t)sz & 0xffu) << 16);
  };
  auto place = [&](float qx, float qy, float qz) {
    const bool lev = __float_as_int(kh) < 0;
    da = nudge(da); db = nudge(db); dc = nudge(dc);   // Q20: the nudged components are the direction from here on
    set_steps(lev);
    const float va = da, vb = db, vc = dc;
    const float ia = rcp_in_range(va), ib = rcp_in_range(vb), ic = rcp_in_range(vc);   // |v| in [1e-30, 1]
    const float Lx = lev ? A.Lx1 : A.Lx, Ly = lev ? A.Ly1 : A.Ly, Lz = lev ? A.Lz1 : A.Lz;
    delx = Lx * fabsf(ia); dely = Ly * fabsf(ib); delz = Lz * fabsf(ic);
    rx = ((va > 0.0f ? Lx : 0.0f) - qx) * ia;
    ry = ((vb > 0.0f ? Ly : 0.0f) - qy) * ib;
    rz = ((vc > 0.0f ? Lz : 0.0f) - qz) * ic;
  };
  auto cell_of = [&]() {
    unsigned c;
    if constexpr (kPow2) c = pc;
    else c = ((unsigned)cz * (unsigned)A.ncy + (unsigned)cy) * (unsigned)A.ncx + (unsigned)cx;
    return kBatch ? c + jpt * A.ncell32 : c;
  };
  // the majorant table's word for the cell (cx, cy, cz): the table itself, or (fly) the block's word if the block is
  // merged, else the voxel's own extinction.  Both loads are issued at once; the indices are valid either way.
  auto voxel_word = [&]() {
    unsigned vox;                          // voxel-sized cells: the cell index is the voxel index
    if constexpr (kPow2) vox = pc;
    else vox = ((unsigned)cz * (unsigned)A.ny + (unsigned)cy) * (unsigned)A.nx + (unsigned)cx;
    return __ldg(A.gsum + jpt * (unsigned)A.nz + (unsigned)Z()) + __ldg(A.cloud + vox);
  };
  auto word_at = [&]() {
    if (kBatch && A.fly) {
      unsigned blk;
      if constexpr (kPow2)                 // the three block coordinates straight from the packed index
        blk = ((pc >> (A.shz + A.lmz)) * (unsigned)A.nby + ((pc >> (A.lx + A.lmy)) & ((unsigned)A.nby - 1u))) * (unsigned)A.nbx +
              ((pc >> A.lmx) & ((unsigned)A.nbx - 1u));
      else
        blk = ((unsigned)(cz >> A.lmz) * (unsigned)A.nby + (unsigned)(cy >> A.lmy)) * (unsigned)A.nbx + (unsigned)(cx >> A.lmx);
      const float B = __ldg(A.btab + jpt * A.nblk32 + blk);
      const float k0 = voxel_word();   // (loading it only when the block is not merged was slower: 56.5 against 54.1 ms)
      return (__float_as_int(B) < 0) ? B : k0;
    }
    return __ldg(A.khat + cell_of());
  };
  // §3.14 roulette: below W0/2 survive with probability wq / W0 exactly (32-bit word of the Philox block at
  // counter e | 2^31 against wq) and continue with W0, else end; both branches go to the ledger
  int fate = 0;
  uint32_t term = 0;
  auto roulette = [&](uint32_t where) {
    if (wq >= kW0 / 2) return false;
    const unsigned long long pid = A.first_id + A.index_base + i;
    const uint4 Y = philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), e | 0x80000000u, sid(), A.keys);
    if ((unsigned long long)Y.w < wq) { t_rgain += kW0 - wq; ++t_rkept; wq = kW0; return false; }
    t_rlost += wq; fate = 5; term = where;
    return true;
  };
  auto flush_thread_counters = [&]() {
    unsigned long long v;
    if (kWeighted) {
      if (t_rlost) atomicAdd(&s_cnt[C_ROUL_LOST], t_rlost);
      if (t_rgain) atomicAdd(&s_cnt[C_ROUL_GAINED], t_rgain);
      v = warp_sum(t_rkept);    if (lane == 0 && v) atomicAdd(&s_cnt[C_ROUL_KEPT], v);
    }
    v = warp_sum(t_sc - t_hg);  if (lane == 0 && v) atomicAdd(&s_cnt[C_RAY], v);
    v = warp_sum(t_hg);         if (lane == 0 && v) atomicAdd(&s_cnt[C_HG], v);
    v = warp_sum(t_sfc);        if (lane == 0 && v) atomicAdd(&s_cnt[C_SFC_HITS], v);
    v = warp_sum(t_cells);      if (lane == 0 && v) atomicAdd(&s_cnt[C_CELLS], v);
    v = warp_sum(t_relevel);    if (lane == 0 && v) atomicAdd(&s_cnt[C_RELEVEL], v);
    // null = events - scatters - absorptions; absorptions are counted at the photon's end, so park the
    // (events - scatters) part here and subtract C_ATM_ABS when the block folds its counters
    v = warp_sum(t_ev - t_sc);  if (lane == 0 && v) atomicAdd(&s_cnt[C_NULL], v);
  };

  // ---- SCATTER: phase-function angle, rotation, new distances to the faces (§3.9) ----------------------
  auto scatter_phase = [&]() {
    if (st == ST_SCATTER) {
      const bool lev = __float_as_int(kh) < 0;
      const float qx = local(da, rx, lev ? A.Lx1 : A.Lx), qy = local(db, ry, lev ? A.Ly1 : A.Ly),
                  qz = local(dc, rz, lev ? A.Lz1 : A.Lz);
      float mu, sn;
      if (sg < 1.5f) { sample_hg(sg, u24(sw2), mu, sn); ++t_hg; }
      else           { sample_rayleigh(u24(sw2), mu, sn); }
      float sp, cp;
      sincos_2pi(u24(sw3), sp, cp);
      rotate_dir(da, db, dc, mu, sn, cp, sp);
      place(qx, qy, qz);
      direct = false; ++t_sc;
      st = ST_MOVE;
    }
  };
  // ---- §3.7b change of level at the face of a merged cell, right where MOVE finds it (ax = the axis just crossed;
  //      kh already holds the ENTERED cell's word).  It used to be a parked phase of its own: 3 per photon, batches
  //      of 4-6 lanes, one visit running both directions and often the arrival code too (31 % of the kernel's
  //      instructions, profiles/r2_trace_kernel.md); inline it runs for the 1-2 lanes that need it at that step.
  auto relevel = [&](bool a0, bool a1, bool a2) {   // which axis was crossed
    // The compiler otherwise lifts the cheap parts of both branches (the in-block offsets, the rescaled face
    // spacings) into the MOVE step itself, where every lane pays for them at every crossing: an empty volatile asm
    // that redefines the inputs keeps them in here (5 % of the kernel's instructions, profiles/r2_trace_kernel.md F).
    asm volatile("" : "+f"(delx), "+f"(dely), "+f"(delz));
    if constexpr (kPow2) asm volatile("" : "+r"(pc));
    const bool px = da > 0.0f, py = db > 0.0f, pz = dc > 0.0f;
    if (__float_as_int(kh) < 0) {
      // into a merged cell: distances to ITS faces (n whole cells further on the other two axes),
      // the index becomes its origin
      const int ox = X() & (A.mx - 1), oy = Y() & (A.my - 1), oz = Z() & (A.mz - 1);   // powers of two
      const float fx = (float)A.mx, fy = (float)A.my, fz = (float)A.mz;
      rx = a0 ? delx * fx : fmaf((float)(px ? A.mx - 1 - ox : ox), delx, rx);
      ry = a1 ? dely * fy : fmaf((float)(py ? A.my - 1 - oy : oy), dely, ry);
      rz = a2 ? delz * fz : fmaf((float)(pz ? A.mz - 1 - oz : oz), delz, rz);
      delx *= fx; dely *= fy; delz *= fz;       // exact: the factors are powers of two
      if constexpr (kPow2) pc &= A.omask; else { cx -= ox; cy -= oy; cz -= oz; }
      set_steps(true);
    } else {
      // out of a merged cell into single cells: which cell of the entered block on the other two
      // axes (k whole cells before the block's face: r / del = r (|v| (1 / L)), §3.7b), and the distances to that cell's faces
      delx *= A.rmx; dely *= A.rmy; delz *= A.rmz;
      if (a0) { rx = delx; if (!px) add_x(A.mx - 1); }
      else { const int k = min(A.mx - 1, (int)(rx * (fabsf(da) * A.rLx))); rx = fmaxf(0.0f, fmaf(-(float)k, delx, rx)); add_x(px ? A.mx - 1 - k : k); }
      if (a1) { ry = dely; if (!py) add_y(A.my - 1); }
      else { const int k = min(A.my - 1, (int)(ry * (fabsf(db) * A.rLy))); ry = fmaxf(0.0f, fmaf(-(float)k, dely, ry)); add_y(py ? A.my - 1 - k : k); }
      if (a2) { rz = delz; if (!pz) add_z(A.mz - 1); }
      else { const int k = min(A.mz - 1, (int)(rz * (fabsf(dc) * A.rLz))); rz = fmaxf(0.0f, fmaf(-(float)k, delz, rz)); add_z(pz ? A.mz - 1 - k : k); }
      kh = (kBatch && A.fly) ? voxel_word() : __ldg(A.khat + cell_of());   // the single cell's own majorant (sign bit clear)
      set_steps(false);
    }
    ++t_relevel;
  };

  for (;;) {
    // the vote: one warp-wide integer add counts the lanes in each of the five states (6 bits each)
    const unsigned votes = __reduce_add_sync(0xffffffffu, 1u << (6u * st));
    // count >= threshold for all five states at once: adding 32 - threshold to a 6-bit field sets its top bit
    // exactly when the count (<= 32) has reached the threshold, and never carries into the next field
    constexpr unsigned bD = 32u, bM = 32u << 6, bC = 32u << 12, bS = 32u << 18, bB = 32u << 24;
    const unsigned full = (votes + A.vote_bias) & (bD | bM | bC | bS | bB);

    if (!exhausted && (full & bD)) {
      // ---- regeneration: hand photon ids to the idle lanes -------------------------------------
      unsigned waiting = __ballot_sync(0xffffffffu, st == ST_DEAD);
      bool got = false;
#pragma unroll 1
      for (int pass = 0; pass < 2 && waiting; ++pass) {
        const unsigned long long have = pool_end - pool_next;
        const unsigned rank = __popc(waiting & lt_mask);
        const bool mine = ((waiting >> lane) & 1u) && (unsigned long long)rank < have;
        if (mine) { i = pool_next + rank; got = true; }
        const unsigned took = __ballot_sync(0xffffffffu, mine);
        pool_next += __popc(took);
        waiting &= ~took;
        if (waiting && pass == 0) {
          unsigned long long base = 0;
          if (lane == 0) base = atomicAdd(A.next_photon, (unsigned long long)A.chunk);
          base = __shfl_sync(0xffffffffu, base, 0);
          pool_next = base < A.n_photons ? base : A.n_photons;
          pool_end = (base + A.chunk < A.n_photons) ? base + A.chunk : A.n_photons;
          if (pool_next > pool_end) pool_next = pool_end;
        }
      }
      if (waiting) exhausted = true;
      if (__any_sync(0xffffffffu, t_ev > (1u << 30) || t_cells > (1u << 30))) {
        flush_thread_counters();                   // keep the 32-bit running totals far from overflow
        if (kRecords) { b_ev -= t_ev; b_sc -= t_sc; b_sfc -= t_sfc; }
        t_ev = t_sc = t_hg = t_sfc = t_cells = t_relevel = 0;
        t_rlost = t_rgain = 0; t_rkept = 0;
      }
      if (got) {
        // ---- §3.6 launch, event index 0 ------------------------------------------------------
        unsigned long long n_full = A.n_full;
        if (kBatch) {
          // which point owns launch index i: last j with offsets[j] <= i
          ig = i;
          int lo = 0, hi = A.n_points;
          while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(A.offsets + mid) <= i) lo = mid; else hi = mid;
          }
          jpt = (uint32_t)(lo + A.first_point);
          i -= __ldg(A.offsets + lo);
          n_full = __ldg(A.nfull + lo);
        }
        const unsigned long long ij = A.index_base + i;   // index in the job: column and pass
        const unsigned long long pid = A.first_id + ij;
        const uint4 X = philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), 0u, sid(), A.keys);
        int ix, iy;
        float e0 = u24(X.x), e1 = u24(X.y);   // sub-pixel entry point
        if (ij < n_full) {
          // column = index mod ncol; 32-bit arithmetic whenever the index allows it
          const uint32_t col = (ij >> 32) ? (uint32_t)(ij % A.ncol) : (uint32_t)ij % (uint32_t)A.ncol;
          ix = (int)(col % (uint32_t)A.nx);
          iy = (int)(col / (uint32_t)A.nx);
          if (A.sobol) {
            // §3.15: point k = pass number of the 2-D Sobol sequence, XORed with the column's digital shift
            const uint32_t k = (ij >> 32) ? (uint32_t)(ij / A.ncol) : (uint32_t)ij / (uint32_t)A.ncol;
            const uint4 S = philox4x32_10(col, sid(), (uint32_t)A.first_id, (uint32_t)(A.first_id >> 32),
                                          A.keys_sobol);
            uint32_t x1 = __brev(k), x2 = 0, V = 0x80000000u;
            for (uint32_t kk = k; kk; kk >>= 1) { if (kk & 1u) x2 ^= V; V ^= V >> 1; }
            e0 = u24(x1 ^ S.x); e1 = u24(x2 ^ S.y);
          }
        } else {
          ix = min((int)(u24(X.z) * (float)A.nx), A.nx - 1);
          iy = min((int)(u24(X.w) * (float)A.ny), A.ny - 1);
        }
        set_cell(ix / A.bx, iy / A.by, A.ncz - 1);
        da = A.sun_x; db = A.sun_y; dc = A.sun_z;
        // §3.5b: the sign bit of the stored majorant marks the cells of a merged cell
        kh = word_at();
        const bool lev = __float_as_int(kh) < 0;
        set_steps(lev);
        int wx = A.bx, wy = A.by;             // cell extent in voxels at this level
        float Lx = A.Lx, Ly = A.Ly, Lz = A.Lz;
        if (lev) {
          if constexpr (kPow2) pc &= A.omask;         // merged-cell origin (factors are powers of two)
          else { cx &= -A.mx; cy &= -A.my; cz &= -A.mz; }
          wx *= A.mx; wy *= A.my; Lx = A.Lx1; Ly = A.Ly1; Lz = A.Lz1;
        }
        const float qx = ((float)(ix % wx) + e0) * A.dx, qy = ((float)(iy % wy) + e1) * A.dy;
        direct = true;
        if (A.diffuse_fraction > 0.0f) {
          // §3.15: block (id, 0 | 2^31): word 0 decides, words 1, 2 give a cosine-weighted downward direction
          const uint4 D = philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), 0x80000000u, sid(), A.keys);
          if (u24(D.x) < A.diffuse_fraction) {
            const float v1 = u24(D.y);
            const float mu = sqrtf(1.0f - v1), sn = sqrtf(v1);
            float sp, cp;
            sincos_2pi(u24(D.z), sp, cp);
            da = sn * cp; db = sn * sp; dc = -mu;
            direct = false;
          }
        }
        if (direct) {
          // place() with the beam's host-computed reciprocals (same IEEE operations)
          delx = Lx * fabsf(A.sun_ix); dely = Ly * fabsf(A.sun_iy); delz = Lz * fabsf(A.sun_iz);
          rx = ((A.sun_ix > 0.0f ? Lx : 0.0f) - qx) * A.sun_ix;
          ry = ((A.sun_iy > 0.0f ? Ly : 0.0f) - qy) * A.sun_iy;
          rz = ((A.sun_iz > 0.0f ? Lz : 0.0f) - Lz) * A.sun_iz;
        } else {
          place(qx, qy, Lz);
        }
        wq = kW0;
        e = 1;
        if (kRecords) { b_ev = t_ev; b_sc = t_sc; b_sfc = t_sfc; }
        draw();
        st = ST_MOVE;
      }
      continue;
    }
    if ((votes & 63u) == 32u) break;

    // a lane moves and no parked phase has reached its batch size
    if ((full & (bM | bC | bS | bB)) == bM) {
      // ---- MOVE: nearest face of the current cell (ties x < y < z), then cross or park (§3.7) -------
      // (rolled loop: one copy of the step and of the level change; the kernel is larger than the instruction cache)
#pragma unroll 1
      for (int rep = A.move_steps; st == ST_MOVE && rep > 0; --rep) {   // a lane leaves the loop with its last MOVE step
      {
        const bool ax0 = (rx <= ry) && (rx <= rz);
        const bool ax1 = !ax0 && (ry <= rz);
        const bool ax2 = !ax0 && !ax1;
        const float t = ax0 ? rx : (ax1 ? ry : rz);
        const float dtau = fabsf(kh) * t;
        if (fabsf(kh) > 0.0f && tau <= dtau) {
          st = ST_COLLIDE;                           // the tentative collision comes first
        } else {
          // leave the cell through that face, carrying the residual optical depth
          tau = tau - dtau;
          ++t_cells;
          rx = ax0 ? delx : rx - t;
          ry = ax1 ? dely : ry - t;
          rz = ax2 ? delz : rz - t;
          // step the cell index; x and y wrap (periodic)
          bool outside;
          if constexpr (kPow2) {
            // one add in the crossed axis' field; the field mask is the periodic wrap in x and y, and in z (the top
            // field) a step out of the domain gives an index >= ncell
            const uint32_t d = ax0 ? dpx : (ax1 ? dpy : dpz);
            const uint32_t m = ax0 ? A.xmask : (ax1 ? A.ymask : A.zmask);
            pc = (pc & ~m) | ((pc + d) & m);
            outside = pc >= A.ncell32;
          } else {
            const int sx = (int)(stp << 24) >> 24, sy = (int)(stp << 16) >> 24, sz = (int)(stp << 8) >> 24;
            if (ax0) { cx += sx; cx = (cx >= A.ncx) ? cx - A.ncx : cx; cx = (cx < 0) ? cx + A.ncx : cx; }
            if (ax1) { cy += sy; cy = (cy >= A.ncy) ? cy - A.ncy : cy; cy = (cy < 0) ? cy + A.ncy : cy; }
            if (ax2) cz += sz;
            outside = (unsigned)cz >= (unsigned)A.ncz;
          }
          if (outside) st = ST_BOUNDARY;             // surface (cz < 0) or domain top
          else {
            const float raw = word_at();
            const bool other = (__float_as_int(raw) ^ __float_as_int(kh)) < 0;   // §3.7b: the entered cell is at the other level
            kh = raw;
            if (other) relevel(ax0, ax1, ax2);
          }
        }
      }
      }
      continue;
    }

    // which parked phase: one that reached its batch size, or (nothing moves) the fullest one
    int phase;
    if (!(full & bM)) {                            // nothing can move
      const unsigned nC = (votes >> 12) & 63u, nS = (votes >> 18) & 63u, nB = (votes >> 24) & 63u;
      phase = (nC >= nS && nC >= nB) ? ST_COLLIDE : (nS >= nB ? ST_SCATTER : ST_BOUNDARY);
    } else {
      phase = (full & bC) ? ST_COLLIDE : ((full & bS) ? ST_SCATTER : ST_BOUNDARY);
    }

    unsigned long long* tally_a;            // arrival / terminal bin
    unsigned long long* tally_b;            // surface absorption after an arrival tally
    if (phase == ST_SCATTER) {
    scatter:
      scatter_phase();
      continue;
    }

    fate = 0;
    term = 0;
    tally_a = nullptr;
    tally_b = nullptr;
    if (phase == ST_COLLIDE) {
      // ---- COLLIDE: fetch the voxel, classify, draw the next event (§3.8) --------------------------
      if (st == ST_COLLIDE) {
        const bool lev = __float_as_int(kh) < 0;
        const float rk = 1.0f / fabsf(kh);
        const float s = tau * rk;
        rx = fmaxf(0.0f, rx - s); ry = fmaxf(0.0f, ry - s); rz = fmaxf(0.0f, rz - s);
        // 32-bit indices: rt_create_grid refuses grids of 2^32 voxels or more
        unsigned vox;
        int vz;
        if (A.unit && !lev) {                         // voxel-sized cell: the cell index is the voxel index
          vz = Z();
          if constexpr (kPow2) vox = pc;
          else vox = ((unsigned)cz * (unsigned)A.ny + (unsigned)cy) * (unsigned)A.nx + (unsigned)cx;
        } else {
          const float qx = local(da, rx, lev ? A.Lx1 : A.Lx), qy = local(db, ry, lev ? A.Ly1 : A.Ly),
                      qz = local(dc, rz, lev ? A.Lz1 : A.Lz);
          const int lx = min((int)(qx * A.rdx), (lev ? A.mx * A.bx : A.bx) - 1);
          const int ly = min((int)(qy * A.rdy), (lev ? A.my * A.by : A.by) - 1);
          const int lz = min((int)(qz * A.rdz), (lev ? A.mz * A.bz : A.bz) - 1);
          vz = Z() * A.bz + lz;
          vox = ((unsigned)vz * (unsigned)A.ny + (unsigned)(Y() * A.by + ly)) * (unsigned)A.nx + (unsigned)(X() * A.bx + lx);
        }
        float4 v;
        if (kBatch && A.cloud) {
          const float kc = __ldg(A.cloud + vox);
          const int z = vz;
          const float ka = __ldg(A.gas + (size_t)jpt * 2u * (unsigned)A.nz + z);
          const float kr = __ldg(A.gas + (size_t)jpt * 2u * (unsigned)A.nz + (unsigned)A.nz + z);
          const float2 pp = __ldg(A.point_par + jpt);
          const float k = (ka + kr) + kc;                                     // §3.4b
          const float w = (k > 0.0f) ? (kr + pp.x * kc) / k : 0.0f;
          float c1 = (1.0f - w) * k;                                          // §3.4
          const float frac = (k > 0.0f) ? kc / k : 0.0f;
          float c2 = c1 + (w * k) * frac;
          c2 = fminf(c2, k);
          c1 = fminf(c1, c2);
          v = make_float4(c1, c2, k, pp.y);
        } else {
          v = __ldg(&A.optics[kBatch ? vox + jpt * A.nvox32 : vox]);
        }
        ++t_ev;
        float xi = u1 * fabsf(kh);
        st = ST_MOVE;
        if (kWeighted) {
          // §3.14: deposit wq * P(absorbed), P = c1 / k_hat as a 24-bit fixed-point number; the rest goes on
          const float f = v.x * rk;
          const unsigned long long pq = min(1u << 24, (unsigned)(f * 16777216.0f));
          const unsigned long long a = (wq * pq) >> 24;
          // one reduction per tentative collision.  Summing consecutive deposits into the same voxel in registers
          // first was measured slower (95.7 -> 101.7 ms on config 3: three more registers spill, profiles/r2_trace_kernel.md)
          if (a) atomicAdd(A.atm_abs + vox, a);
          if (a && direct && A.atm_dir) atomicAdd(A.atm_dir + vox, a);
          wq -= a;
          if (wq == 0) { fate = 1; term = (uint32_t)vox; }
          xi = fmaf(u1, fabsf(kh) - v.x, v.x);      // what happens instead: uniform on [c1, k_hat)
        } else if (xi < v.x) {                      // absorbed by the gas / droplet
          tally_a = A.atm_abs + vox;
          if (direct && A.atm_dir) atomicAdd(A.atm_dir + vox, kW0);
          fate = 1; term = (uint32_t)vox;
        }
        if (fate == 0) {
          if (xi < v.z) {                           // real scattering: angle and rotation in SCATTER
            st = ST_SCATTER;
            sg = (xi < v.y) ? v.w : 2.0f;
            sw2 = w2; sw3 = w3;
          }
          if (kWeighted && roulette((uint32_t)vox)) {
            if (st == ST_SCATTER) { ++t_sc; if (sg < 1.5f) ++t_hg; }   // the event itself is still counted
          } else {
            ++e;
            if (e > kEventCap) {                    // §3.12 (the capped event itself is still counted)
              if (st == ST_SCATTER) { ++t_sc; if (sg < 1.5f) ++t_hg; }
              fate = 4; term = 0;
            } else {
              draw();
            }
          }
        }
      }
    } else {
      // ---- BOUNDARY: arrival at the surface (§3.10) or exit through the domain top (§3.11) ---------------
      if (st == ST_BOUNDARY) {
        const bool lev = __float_as_int(kh) < 0;
        const float qx = local(da, rx, lev ? A.Lx1 : A.Lx), qy = local(db, ry, lev ? A.Ly1 : A.Ly);
        const int hx = X() * A.bx + min((int)(qx * A.rdx), (lev ? A.mx * A.bx : A.bx) - 1);
        const int hy = Y() * A.by + min((int)(qy * A.rdy), (lev ? A.my * A.by : A.by) - 1);
        const unsigned col = (unsigned)hy * (unsigned)A.nx + (unsigned)hx;
        if (Z() >= 0) {                             // left through the domain top
          if (kWeighted) atomicAdd(A.toa_up + col, wq); else tally_a = A.toa_up + col;
          fate = 3; term = (uint32_t)col;
        } else {                                    // Lambertian surface
          ++t_sfc;
          bool reflect;
          if (kWeighted) {
            // §3.14: arrival tallied with the weight; the albedo reduces the weight, 24-bit fixed point
            atomicAdd((direct ? A.sfc_dir : A.sfc_dif) + col, wq);
            const unsigned long long aq = min(1u << 24, (unsigned)(__ldg(&A.albedo[kBatch ? col + jpt * A.ncol32 : col]) * 16777216.0f));
            const unsigned long long refl = (wq * aq) >> 24;
            if (wq - refl) atomicAdd(A.sfc_abs + col, wq - refl);
            wq = refl;
            if (wq == 0) { fate = 2; term = (uint32_t)col; reflect = false; }
            else reflect = !roulette((uint32_t)col);
          } else {
            tally_a = (direct ? A.sfc_dir : A.sfc_dif) + col;
            reflect = u1 < __ldg(&A.albedo[kBatch ? col + jpt * A.ncol32 : col]);
            if (!reflect) { tally_b = A.sfc_abs + col; fate = 2; term = (uint32_t)col; }
          }
          if (reflect) {
            const float u2 = u24(w2);
            const float mu = sqrtf(1.0f - u2), sn = sqrtf(u2);
            float sp, cp;
            sincos_2pi(u24(w3), sp, cp);
            da = sn * cp; db = sn * sp; dc = mu;
            direct = false;                         // back in the cell it left (cz = 0): same level, same majorant
            if constexpr (kPow2) pc &= ~A.zmask; else cz = 0;
            place(qx, qy, 0.0f);
            ++e;
            if (e > kEventCap) { fate = 4; term = 0; }   // §3.12
            else {
              draw();
              st = ST_MOVE;
            }
          }
        }
      }
    }
    if (fate != 0) st = ST_DEAD;

    // ---- tallies (converged): warp-aggregated 64-bit integer atomics -----------------------------
    {
      const unsigned ma = __ballot_sync(0xffffffffu, tally_a != nullptr);
      if (ma) {
        if (tally_a) tally_add(ma, tally_a);
        const unsigned mb = __ballot_sync(0xffffffffu, tally_b != nullptr);
        if (mb && tally_b) tally_add(mb, tally_b);
      }
    }
    if (__any_sync(0xffffffffu, fate != 0)) {
      // photons finished: each adds one to its fate's 32-bit counter of the block (a native shared-memory atomic;
      // a few lanes at most share an address), and writes its record
      if (fate != 0) atomicAdd(&s_fate[fate], 1u);
      if (kWeighted && fate == 4) atomicAdd(&s_cnt[C_CAPPED_E], wq);     // rare: a 64-bit shared atomic is a CAS loop
      if (kRecords && fate != 0) {
        uint4 r;
        r.x = (uint32_t)fate | (min(t_sfc - b_sfc, 0xFFFFFFu) << 8);
        r.y = term; r.z = t_ev - b_ev; r.w = t_sc - b_sc;
        reinterpret_cast<uint4*>(A.records)[kBatch ? ig : i] = r;
      }
    }
    // With voxel-sized cells nearly every collision is a scattering, so SCATTER runs right behind COLLIDE without
    // another vote: a jump back to the ONE copy of the phase (a second inlined copy costs more than the vote).
    if (A.unit && phase == ST_COLLIDE) goto scatter;
  }

  flush_thread_counters();
  __syncthreads();
  if (threadIdx.x == 0) {
    s_cnt[C_ATM_ABS] += s_fate[1]; s_cnt[C_SFC_ABS] += s_fate[2]; s_cnt[C_TOA] += s_fate[3];
    s_cnt[C_CAPPED] += s_fate[4]; s_cnt[C_ROUL_KILLED] += s_fate[5];
    if (!kWeighted) s_cnt[C_CAPPED_E] += kW0 * (unsigned long long)s_fate[4];
    s_cnt[C_NULL] -= s_cnt[C_ATM_ABS];   // events - scatters - absorptions
  }
  __syncthreads();
  if (threadIdx.x < C_COUNT && s_cnt[threadIdx.x] != 0ull)
    atomicAdd(&A.counters[threadIdx.x], s_cnt[threadIdx.x]);
}

}  // namespace rt
