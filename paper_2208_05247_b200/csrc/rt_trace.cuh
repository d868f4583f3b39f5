// rt_trace.cuh — the persistent photon-tracing kernel.
//
// One thread carries one photon at a time.  Its position inside the current acceleration cell is held
// as the remaining distances (rx, ry, rz) along the flight direction to the cell's next face on each
// axis: a cell crossing is ~25 instructions (smallest of three, two subtractions, one
// reset to the face spacing, index step, one 4-byte load of the majorant), a null collision updates the
// three distances and nothing else.  With cheap crossings a fine acceleration grid (2^3 voxels per
// cell) pays: 38 tentative collisions and 168 crossings per photon on the 512x512x128 cumulus field
// instead of 202 and 42 with 8^3 cells.
//
// Divergence.  MOVE (cross or collide) is what every live lane does each iteration.  A real scatter
// (phase-function inversion, rotation, three IEEE divisions: ~200 instructions) is chosen by few lanes
// per iteration; run inline it executed in 84 % of the iterations with 2 of 32 lanes active (ncu,
// profiles/r1_baseline_*).  So a lane that chose to scatter parks in SCATTER and the warp runs that
// phase when kScatterBatch lanes wait (ballot/popc vote); DEAD lanes are refilled kRegenBatch at a time
// from a warp-private pool of photon ids taken in chunks from a global counter (BASELINE.json
// north_star: "compacted and regenerated persistently with warp-level ballot/shuffle").  A photon's own
// sequence of arithmetic operations does not depend on the scheduling, so neither do the results.
#pragma once
#include "rt_device.cuh"

namespace rt {

constexpr unsigned long long kW0 = 1ull << 32;  // tally quanta per photon
constexpr uint32_t kEventCap = 1u << 20;        // §3.12
constexpr float kTiny = 1e-30f;                 // direction components are nudged away from 0
constexpr int kTraceThreads = 256;
constexpr int kChunk = 128;                     // photon ids a warp takes per global atomic
#ifndef RT_MIN_BLOCKS
#define RT_MIN_BLOCKS 3
#endif
#ifndef RT_REGEN_BATCH
#define RT_REGEN_BATCH 6
#endif
#ifndef RT_SCATTER_BATCH
#define RT_SCATTER_BATCH 6
#endif
constexpr int kRegenBatch = RT_REGEN_BATCH;       // refill when this many lanes are idle (or nothing else to do)
constexpr int kScatterBatch = RT_SCATTER_BATCH;   // run SCATTER when this many lanes wait for it (or nothing else)

enum Counter { C_NULL = 0, C_RAY, C_HG, C_ATM_ABS, C_SFC_HITS, C_SFC_ABS, C_TOA, C_CAPPED, C_CELLS,
               C_CAPPED_E, C_COUNT };

enum : uint32_t { ST_DEAD = 0, ST_MOVE = 1, ST_SCATTER = 2 };

struct TraceArgs {
  int nx, ny, nz, bx, by, bz, ncx, ncy, ncz;
  float dx, dy, dz, rdx, rdy, rdz, Lx, Ly, Lz;
  float sun_x, sun_y, sun_z, sun_ix, sun_iy, sun_iz;  // beam direction and 1/nudge(component), host-computed
  const float4* __restrict__ optics;   // [z][y][x] (c1, c2, c3, g)
  const float* __restrict__ khat;      // [cz][cy][cx]
  const float* __restrict__ albedo;    // [y][x]
  unsigned long long* atm_abs;         // [z][y][x]
  unsigned long long *sfc_dir, *sfc_dif, *sfc_abs, *toa_up;  // [y][x]
  unsigned long long* counters;        // C_COUNT words
  unsigned long long* next_photon;     // work counter, zeroed before launch
  uint32_t* records;                   // 4 words per photon or nullptr
  unsigned long long n_photons, first_id, n_full, ncol;
  uint32_t key0, key1, stream_id;
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



template <bool kRecords>
__global__ void __launch_bounds__(kTraceThreads, RT_MIN_BLOCKS) trace_kernel(const TraceArgs A) {
  __shared__ unsigned long long s_cnt[C_COUNT];
  if (threadIdx.x < C_COUNT) s_cnt[threadIdx.x] = 0ull;
  __syncthreads();

  const unsigned lane = threadIdx.x & 31u;
  const unsigned lt_mask = (1u << lane) - 1u;
  unsigned long long pool_next = 0, pool_end = 0;  // warp-uniform chunk of photon indices
  bool exhausted = false;                          // warp-uniform: the global counter has run out

  // photon state
  uint32_t st = ST_DEAD;
  unsigned long long i = 0;
  uint32_t e = 0;
  int cx = 0, cy = 0, cz = 0;
  float da = 0, db = 0, dc = -1;          // unit direction
  float rx = 0, ry = 0, rz = 0;           // remaining distance to the cell's next face on each axis
  float delx = 0, dely = 0, delz = 0;     // distance between successive faces on each axis
  float tau = 0, kh = 0, u1 = 0;
  uint32_t w2 = 0, w3 = 0;                // words 2, 3 of the current event's draw
  uint32_t sw2 = 0, sw3 = 0;              // ... of the event that chose SCATTER (its draw is already replaced)
  float sg = 0;                           // asymmetry parameter for the pending scatter; 2 = Rayleigh
  bool direct = true;
  // event counts: running totals of this thread; a photon's own counts are differences (records)
  uint32_t t_ev = 0, t_sc = 0, t_hg = 0, t_sfc = 0, t_cells = 0;
  uint32_t b_ev = 0, b_sc = 0, b_sfc = 0;  // totals when the current photon was launched (records only)

  auto draw = [&]() {
    const unsigned long long pid = A.first_id + i;
    const uint4 X = philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), e, A.stream_id, A.key0, A.key1);
    tau = neg_log(1.0f - u24(X.x)); u1 = u24(X.y); w2 = X.z; w3 = X.w;
  };
  // local coordinate from a remaining distance: q = face - v r, face = L if v > 0 else 0
  auto local = [&](float d, float r, float L) {
    const float v = nudge(d);
    return fminf(L, fmaxf(0.0f, fmaf(-v, r, v > 0.0f ? L : 0.0f)));
  };
  // after a change of direction at local position (qx, qy, qz): reciprocals, face spacings, distances
  auto place = [&](float qx, float qy, float qz) {
    const float va = nudge(da), vb = nudge(db), vc = nudge(dc);
    const float ia = 1.0f / va, ib = 1.0f / vb, ic = 1.0f / vc;
    delx = A.Lx * fabsf(ia); dely = A.Ly * fabsf(ib); delz = A.Lz * fabsf(ic);
    rx = ((va > 0.0f ? A.Lx : 0.0f) - qx) * ia;
    ry = ((vb > 0.0f ? A.Ly : 0.0f) - qy) * ib;
    rz = ((vc > 0.0f ? A.Lz : 0.0f) - qz) * ic;
  };
  auto flush_thread_counters = [&]() {
    unsigned long long v;
    v = warp_sum(t_sc - t_hg);  if (lane == 0 && v) atomicAdd(&s_cnt[C_RAY], v);
    v = warp_sum(t_hg);         if (lane == 0 && v) atomicAdd(&s_cnt[C_HG], v);
    v = warp_sum(t_sfc);        if (lane == 0 && v) atomicAdd(&s_cnt[C_SFC_HITS], v);
    v = warp_sum(t_cells);      if (lane == 0 && v) atomicAdd(&s_cnt[C_CELLS], v);
    // null = events - scatters - absorptions; absorptions are counted at the photon's end, so park the
    // (events - scatters) part here and subtract C_ATM_ABS when the block folds its counters
    v = warp_sum(t_ev - t_sc);  if (lane == 0 && v) atomicAdd(&s_cnt[C_NULL], v);
  };

  for (;;) {
    const unsigned bM = __ballot_sync(0xffffffffu, st == ST_MOVE);
    const unsigned bS = __ballot_sync(0xffffffffu, st == ST_SCATTER);
    const unsigned live = bM | bS;
    int fate = 0;
    uint32_t term = 0;
    unsigned long long* tally_a = nullptr;  // arrival / terminal bin
    unsigned long long* tally_b = nullptr;  // surface absorption after an arrival tally

    if (!exhausted && (__popc(~live) >= kRegenBatch || !live)) {
      // ---- regeneration: hand photon ids to the idle lanes -------------------------------------
      unsigned waiting = ~live;
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
          if (lane == 0) base = atomicAdd(A.next_photon, (unsigned long long)kChunk);
          base = __shfl_sync(0xffffffffu, base, 0);
          pool_next = base < A.n_photons ? base : A.n_photons;
          pool_end = (base + kChunk < A.n_photons) ? base + kChunk : A.n_photons;
          if (pool_next > pool_end) pool_next = pool_end;
        }
      }
      if (waiting) exhausted = true;
      if (__any_sync(0xffffffffu, t_ev > (1u << 30) || t_cells > (1u << 30))) {
        flush_thread_counters();                   // keep the 32-bit running totals far from overflow
        if (kRecords) { b_ev -= t_ev; b_sc -= t_sc; b_sfc -= t_sfc; }
        t_ev = t_sc = t_hg = t_sfc = t_cells = 0;
      }
      if (got) {
        // ---- §3.6 launch, event index 0 ------------------------------------------------------
        const unsigned long long pid = A.first_id + i;
        const uint4 X = philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), 0u, A.stream_id, A.key0, A.key1);
        int ix, iy;
        if (i < A.n_full) {
          // column = i mod ncol; 32-bit arithmetic whenever the index allows it
          const uint32_t col = (i >> 32) ? (uint32_t)(i % A.ncol) : (uint32_t)i % (uint32_t)A.ncol;
          ix = (int)(col % (uint32_t)A.nx);
          iy = (int)(col / (uint32_t)A.nx);
        } else {
          ix = min((int)(u24(X.z) * (float)A.nx), A.nx - 1);
          iy = min((int)(u24(X.w) * (float)A.ny), A.ny - 1);
        }
        cx = ix / A.bx; cy = iy / A.by; cz = A.ncz - 1;
        da = A.sun_x; db = A.sun_y; dc = A.sun_z;
        // place() with the beam's host-computed reciprocals (same IEEE operations)
        delx = A.Lx * fabsf(A.sun_ix); dely = A.Ly * fabsf(A.sun_iy); delz = A.Lz * fabsf(A.sun_iz);
        rx = ((A.sun_ix > 0.0f ? A.Lx : 0.0f) - ((float)(ix % A.bx) + u24(X.x)) * A.dx) * A.sun_ix;
        ry = ((A.sun_iy > 0.0f ? A.Ly : 0.0f) - ((float)(iy % A.by) + u24(X.y)) * A.dy) * A.sun_iy;
        rz = ((A.sun_iz > 0.0f ? A.Lz : 0.0f) - A.Lz) * A.sun_iz;
        direct = true;
        e = 1;
        if (kRecords) { b_ev = t_ev; b_sc = t_sc; b_sfc = t_sfc; }
        draw();
        kh = __ldg(&A.khat[((size_t)cz * A.ncy + cy) * A.ncx + cx]);
        st = ST_MOVE;
      }
      continue;
    }
    if (!live) break;

    if (__popc(bS) >= kScatterBatch || !bM) {
      // ---- SCATTER: phase-function angle, rotation, new distances to the faces (§3.9) --------------
      if (st == ST_SCATTER) {
        const float qx = local(da, rx, A.Lx), qy = local(db, ry, A.Ly), qz = local(dc, rz, A.Lz);
        float mu;
        if (sg < 1.5f) { mu = sample_hg(sg, u24(sw2)); ++t_hg; }
        else           { mu = sample_rayleigh(u24(sw2)); }
        float sp, cp;
        sincos_2pi(u24(sw3), sp, cp);
        rotate_dir(da, db, dc, mu, cp, sp);
        place(qx, qy, qz);
        direct = false; ++t_sc;
        st = ST_MOVE;
      }
    } else if (st == ST_MOVE) {
      // ---- MOVE: nearest face of the current cell (ties x < y < z), then collide or cross (§3.7) ----
      int axis; float t;
      if (rx <= ry && rx <= rz) { axis = 0; t = rx; }
      else if (ry <= rz)        { axis = 1; t = ry; }
      else                      { axis = 2; t = rz; }
      const float dtau = kh * t;
      if (kh > 0.0f && tau <= dtau) {
        // §3.8 tentative collision inside this cell: fetch the voxel, classify, draw the next event
        const float s = tau * (1.0f / kh);
        rx = fmaxf(0.0f, rx - s); ry = fmaxf(0.0f, ry - s); rz = fmaxf(0.0f, rz - s);
        const float qx = local(da, rx, A.Lx), qy = local(db, ry, A.Ly), qz = local(dc, rz, A.Lz);
        const int lx = min((int)(qx * A.rdx), A.bx - 1);
        const int ly = min((int)(qy * A.rdy), A.by - 1);
        const int lz = min((int)(qz * A.rdz), A.bz - 1);
        const size_t vox = ((size_t)(cz * A.bz + lz) * A.ny + (cy * A.by + ly)) * A.nx + (cx * A.bx + lx);
        const float4 v = __ldg(&A.optics[vox]);
        ++t_ev;
        const float xi = u1 * kh;
        if (xi < v.x) {                             // absorbed by the gas / droplet
          tally_a = A.atm_abs + vox;
          fate = 1; term = (uint32_t)vox;
        } else {
          if (xi < v.z) {                           // real scattering: angle and rotation in SCATTER
            st = ST_SCATTER;
            sg = (xi < v.y) ? v.w : 2.0f;
            sw2 = w2; sw3 = w3;
          }
          ++e;
          if (e > kEventCap) {                      // §3.12 (the capped event itself is still counted)
            if (st == ST_SCATTER) { ++t_sc; if (sg < 1.5f) ++t_hg; }
            fate = 4; term = 0;
          } else {
            draw();
          }
        }
      } else {
        // §3.7 leave the cell through `axis`, carrying the residual optical depth
        tau = tau - dtau;
        ++t_cells;
        bool at_sfc = false, at_top = false;
        if (axis == 0) {
          ry = ry - t; rz = rz - t; rx = delx;
          if (nudge(da) > 0.0f) { ++cx; if (cx == A.ncx) cx = 0; }
          else                  { --cx; if (cx < 0) cx = A.ncx - 1; }
        } else if (axis == 1) {
          rx = rx - t; rz = rz - t; ry = dely;
          if (nudge(db) > 0.0f) { ++cy; if (cy == A.ncy) cy = 0; }
          else                  { --cy; if (cy < 0) cy = A.ncy - 1; }
        } else {
          rx = rx - t; ry = ry - t; rz = delz;
          if (nudge(dc) > 0.0f) { ++cz; at_top = (cz == A.ncz); }
          else                  { --cz; at_sfc = (cz < 0); }
        }
        if (at_sfc || at_top) {
          const float qx = local(da, rx, A.Lx), qy = local(db, ry, A.Ly);
          const int hx = cx * A.bx + min((int)(qx * A.rdx), A.bx - 1);
          const int hy = cy * A.by + min((int)(qy * A.rdy), A.by - 1);
          const size_t col = (size_t)hy * A.nx + hx;
          if (at_top) {                             // §3.11 leaves through the domain top
            tally_a = A.toa_up + col;
            fate = 3; term = (uint32_t)col;
          } else {                                  // §3.10 Lambertian surface
            ++t_sfc;
            tally_a = (direct ? A.sfc_dir : A.sfc_dif) + col;
            if (u1 < __ldg(&A.albedo[col])) {
              const float u2 = u24(w2);
              const float mu = sqrtf(1.0f - u2), sn = sqrtf(u2);
              float sp, cp;
              sincos_2pi(u24(w3), sp, cp);
              da = sn * cp; db = sn * sp; dc = mu;
              direct = false; cz = 0;
              place(qx, qy, 0.0f);
              ++e;
              if (e > kEventCap) { fate = 4; term = 0; }   // §3.12
              else draw();
            } else {
              tally_b = A.sfc_abs + col;
              fate = 2; term = (uint32_t)col;
            }
          }
        }
        if (fate == 0) kh = __ldg(&A.khat[((size_t)cz * A.ncy + cy) * A.ncx + cx]);
      }
      if (fate != 0) st = ST_DEAD;
    }

    // ---- tallies (converged): warp-aggregated 64-bit integer atomics -----------------------------
    const unsigned ma = __ballot_sync(0xffffffffu, tally_a != nullptr);
    if (ma) {
      if (tally_a) tally_add(ma, tally_a);
      const unsigned mb = __ballot_sync(0xffffffffu, tally_b != nullptr);
      if (mb && tally_b) tally_add(mb, tally_b);
    }
    if (__any_sync(0xffffffffu, fate != 0)) {
      // photons finished: count their fates per warp, write their records
      const unsigned f1 = __ballot_sync(0xffffffffu, fate == 1), f2 = __ballot_sync(0xffffffffu, fate == 2);
      const unsigned f3 = __ballot_sync(0xffffffffu, fate == 3), f4 = __ballot_sync(0xffffffffu, fate == 4);
      if (lane == 0) {
        if (f1) atomicAdd(&s_cnt[C_ATM_ABS], (unsigned long long)__popc(f1));
        if (f2) atomicAdd(&s_cnt[C_SFC_ABS], (unsigned long long)__popc(f2));
        if (f3) atomicAdd(&s_cnt[C_TOA], (unsigned long long)__popc(f3));
        if (f4) {
          atomicAdd(&s_cnt[C_CAPPED], (unsigned long long)__popc(f4));
          atomicAdd(&s_cnt[C_CAPPED_E], kW0 * (unsigned long long)__popc(f4));
        }
      }
      if (kRecords && fate != 0) {
        uint4 r;
        r.x = (uint32_t)fate | (min(t_sfc - b_sfc, 0xFFFFFFu) << 8);
        r.y = term; r.z = t_ev - b_ev; r.w = t_sc - b_sc;
        reinterpret_cast<uint4*>(A.records)[i] = r;
      }
    }
  }

  flush_thread_counters();
  __syncthreads();
  if (threadIdx.x == 0) s_cnt[C_NULL] -= s_cnt[C_ATM_ABS];   // events - scatters - absorptions
  __syncthreads();
  if (threadIdx.x < C_COUNT && s_cnt[threadIdx.x] != 0ull)
    atomicAdd(&A.counters[threadIdx.x], s_cnt[threadIdx.x]);
}

}  // namespace rt
