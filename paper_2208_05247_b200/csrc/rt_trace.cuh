// rt_trace.cuh — the persistent photon-tracing kernel.
// One thread carries one photon at a time; a warp draws photon ids in chunks from a global
// counter and refills idle lanes with ballot/popc so lanes stay busy through the long tail of
// in-cloud photons (BASELINE.json north_star: "compacted and regenerated persistently").
#pragma once
#include "rt_device.cuh"

namespace rt {

constexpr unsigned long long kW0 = 1ull << 32;  // tally quanta per photon
constexpr uint32_t kEventCap = 1u << 20;        // §3.12
constexpr float kTiny = 1e-30f;                 // direction components are nudged away from 0
constexpr int kTraceThreads = 256;
constexpr int kChunk = 128;                     // photon ids a warp takes per global atomic

enum Counter { C_NULL = 0, C_RAY, C_HG, C_ATM_ABS, C_SFC_HITS, C_SFC_ABS, C_TOA, C_CAPPED, C_CELLS,
               C_CAPPED_E, C_COUNT };

struct TraceArgs {
  int nx, ny, nz, bx, by, bz, ncx, ncy, ncz;
  float dx, dy, dz, rdx, rdy, rdz, Lx, Ly, Lz;
  float sun_x, sun_y, sun_z;
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

template <bool kRecords>
__global__ void __launch_bounds__(kTraceThreads) trace_kernel(const TraceArgs A) {
  __shared__ unsigned long long s_cnt[C_COUNT];
  if (threadIdx.x < C_COUNT) s_cnt[threadIdx.x] = 0ull;
  __syncthreads();

  const unsigned lane = threadIdx.x & 31u;
  const unsigned lt_mask = (1u << lane) - 1u;
  unsigned long long pool_next = 0, pool_end = 0;  // warp-uniform chunk of photon indices
  bool alive = false, exhausted = false;

  // photon state
  unsigned long long i = 0;
  uint32_t p_lo = 0, p_hi = 0, e = 0;
  int cx = 0, cy = 0, cz = 0;
  float qx = 0, qy = 0, qz = 0, da = 0, db = 0, dc = -1, ia = 0, ib = 0, ic = 0;
  float tau = 0, kh = 0, u1 = 0, u2 = 0, u3 = 0;
  bool direct = true;
  uint32_t n_ev = 0, n_sc = 0, n_hg = 0, n_sfc = 0, n_cells = 0;

  for (;;) {
    // ---- regeneration: refill idle lanes (converged) --------------------------------------
    const unsigned need = __ballot_sync(0xffffffffu, !alive && !exhausted);
    if (need) {
      // hand out what the warp's pool has, then take one fresh chunk if lanes are still waiting
      unsigned waiting = need;
#pragma unroll 1
      for (int pass = 0; pass < 2 && waiting; ++pass) {
        const unsigned long long have = pool_end - pool_next;
        const unsigned rank = __popc(waiting & lt_mask);
        const bool mine = ((waiting >> lane) & 1u) && (unsigned long long)rank < have;
        if (mine) { i = pool_next + rank; alive = true; }
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
      if ((waiting >> lane) & 1u) exhausted = true;

      if (((need & ~waiting) >> lane) & 1u) {
        // ---- §3.6 launch, event index 0 -----------------------------------------------------
        const unsigned long long pid = A.first_id + i;
        p_lo = (uint32_t)pid; p_hi = (uint32_t)(pid >> 32);
        uint4 X = philox4x32_10(p_lo, p_hi, 0u, A.stream_id, A.key0, A.key1);
        int ix, iy;
        if (i < A.n_full) {
          const unsigned long long col = i % A.ncol;
          ix = (int)(col % (unsigned long long)A.nx);
          iy = (int)(col / (unsigned long long)A.nx);
        } else {
          ix = min((int)(u24(X.z) * (float)A.nx), A.nx - 1);
          iy = min((int)(u24(X.w) * (float)A.ny), A.ny - 1);
        }
        cx = ix / A.bx; cy = iy / A.by; cz = A.ncz - 1;
        qx = ((float)(ix % A.bx) + u24(X.x)) * A.dx;
        qy = ((float)(iy % A.by) + u24(X.y)) * A.dy;
        qz = A.Lz;
        da = A.sun_x; db = A.sun_y; dc = A.sun_z;
        ia = 1.0f / (fabsf(da) < kTiny ? kTiny : da);
        ib = 1.0f / (fabsf(db) < kTiny ? kTiny : db);
        ic = 1.0f / (fabsf(dc) < kTiny ? kTiny : dc);
        direct = true;
        e = 1; n_ev = n_sc = n_hg = n_sfc = n_cells = 0;
        X = philox4x32_10(p_lo, p_hi, e, A.stream_id, A.key0, A.key1);
        tau = neg_log(1.0f - u24(X.x)); u1 = u24(X.y); u2 = u24(X.z); u3 = u24(X.w);
        kh = __ldg(&A.khat[((size_t)cz * A.ncy + cy) * A.ncx + cx]);
      }
    }
    if (!__any_sync(0xffffffffu, alive)) break;

    // ---- one step of the photon: a cell crossing or a tentative collision ------------------
    int fate = 0;
    uint32_t term = 0;
    unsigned long long* tally_a = nullptr;  // arrival / terminal bin
    unsigned long long* tally_b = nullptr;  // surface absorption after an arrival tally
    if (alive) {
      const float va = fabsf(da) < kTiny ? kTiny : da;
      const float vb = fabsf(db) < kTiny ? kTiny : db;
      const float vc = fabsf(dc) < kTiny ? kTiny : dc;
      // §3.7 distance to the nearest face of the current cell; ties x < y < z
      const float tx = ((va > 0.0f ? A.Lx : 0.0f) - qx) * ia;
      const float ty = ((vb > 0.0f ? A.Ly : 0.0f) - qy) * ib;
      const float tz = ((vc > 0.0f ? A.Lz : 0.0f) - qz) * ic;
      int axis; float t;
      if (tx <= ty && tx <= tz) { axis = 0; t = tx; }
      else if (ty <= tz)        { axis = 1; t = ty; }
      else                      { axis = 2; t = tz; }
      const float dtau = kh * t;
      bool redraw = false;
      if (kh > 0.0f && tau <= dtau) {
        // §3.8 tentative collision inside this cell
        const float s = tau * (1.0f / kh);
        qx = fminf(A.Lx, fmaxf(0.0f, fmaf(va, s, qx)));
        qy = fminf(A.Ly, fmaxf(0.0f, fmaf(vb, s, qy)));
        qz = fminf(A.Lz, fmaxf(0.0f, fmaf(vc, s, qz)));
        const int lx = min((int)(qx * A.rdx), A.bx - 1);
        const int ly = min((int)(qy * A.rdy), A.by - 1);
        const int lz = min((int)(qz * A.rdz), A.bz - 1);
        const size_t vox = ((size_t)(cz * A.bz + lz) * A.ny + (cy * A.by + ly)) * A.nx + (cx * A.bx + lx);
        const float4 v = __ldg(&A.optics[vox]);
        ++n_ev;
        const float xi = u1 * kh;
        if (xi < v.x) {                         // absorbed by the gas / droplet
          tally_a = A.atm_abs + vox;
          fate = 1; term = (uint32_t)vox;
        } else if (xi < v.z) {                  // real scattering
          float mu;
          if (xi < v.y) { mu = sample_hg(v.w, u2); ++n_hg; }
          else          { mu = sample_rayleigh(u2); }
          float sp, cp;
          sincos_2pi(u3, sp, cp);
          rotate_dir(da, db, dc, mu, cp, sp);
          ia = 1.0f / (fabsf(da) < kTiny ? kTiny : da);
          ib = 1.0f / (fabsf(db) < kTiny ? kTiny : db);
          ic = 1.0f / (fabsf(dc) < kTiny ? kTiny : dc);
          direct = false; ++n_sc;
        }
        if (fate == 0) redraw = true;
      } else {
        // §3.7 leave the cell through `axis`, carrying the residual optical depth
        tau = tau - dtau;
        qx = fminf(A.Lx, fmaxf(0.0f, fmaf(va, t, qx)));
        qy = fminf(A.Ly, fmaxf(0.0f, fmaf(vb, t, qy)));
        qz = fminf(A.Lz, fmaxf(0.0f, fmaf(vc, t, qz)));
        ++n_cells;
        bool at_sfc = false, at_top = false;
        if (axis == 0) {
          if (va > 0.0f) { ++cx; if (cx == A.ncx) cx = 0; qx = 0.0f; }
          else           { --cx; if (cx < 0) cx = A.ncx - 1; qx = A.Lx; }
        } else if (axis == 1) {
          if (vb > 0.0f) { ++cy; if (cy == A.ncy) cy = 0; qy = 0.0f; }
          else           { --cy; if (cy < 0) cy = A.ncy - 1; qy = A.Ly; }
        } else {
          if (vc > 0.0f) { ++cz; qz = 0.0f; at_top = (cz == A.ncz); }
          else           { --cz; qz = A.Lz; at_sfc = (cz < 0); }
        }
        if (at_sfc || at_top) {
          const int hx = cx * A.bx + min((int)(qx * A.rdx), A.bx - 1);
          const int hy = cy * A.by + min((int)(qy * A.rdy), A.by - 1);
          const size_t col = (size_t)hy * A.nx + hx;
          if (at_top) {                         // §3.11 leaves through the domain top
            tally_a = A.toa_up + col;
            fate = 3; term = (uint32_t)col;
          } else {                              // §3.10 Lambertian surface
            ++n_sfc;
            tally_a = (direct ? A.sfc_dir : A.sfc_dif) + col;
            if (u1 < __ldg(&A.albedo[col])) {
              const float mu = sqrtf(1.0f - u2), s = sqrtf(u2);
              float sp, cp;
              sincos_2pi(u3, sp, cp);
              da = s * cp; db = s * sp; dc = mu;
              ia = 1.0f / (fabsf(da) < kTiny ? kTiny : da);
              ib = 1.0f / (fabsf(db) < kTiny ? kTiny : db);
              ic = 1.0f / (fabsf(dc) < kTiny ? kTiny : dc);
              direct = false; cz = 0; qz = 0.0f;
              redraw = true;
            } else {
              tally_b = A.sfc_abs + col;
              fate = 2; term = (uint32_t)col;
            }
          }
        }
        if (fate == 0) kh = __ldg(&A.khat[((size_t)cz * A.ncy + cy) * A.ncx + cx]);
      }
      if (redraw) {
        ++e;
        if (e > kEventCap) {                    // §3.12
          fate = 4; term = 0;
        } else {
          const uint4 X = philox4x32_10(p_lo, p_hi, e, A.stream_id, A.key0, A.key1);
          tau = neg_log(1.0f - u24(X.x)); u1 = u24(X.y); u2 = u24(X.z); u3 = u24(X.w);
        }
      }
    }

    // ---- tallies (converged): warp-aggregated 64-bit integer atomics ----------------------------
    const unsigned ma = __ballot_sync(0xffffffffu, tally_a != nullptr);
    if (ma) {
      if (tally_a) tally_add(ma, tally_a);
      const unsigned mb = __ballot_sync(0xffffffffu, tally_b != nullptr);
      if (mb && tally_b) tally_add(mb, tally_b);
    }
    if (fate != 0) {
      // photon finished: fold its event counts into the block counters, write its record
      const uint32_t n_abs = (fate == 1) ? 1u : 0u;
      atomicAdd(&s_cnt[C_NULL], (unsigned long long)(n_ev - n_sc - n_abs));
      atomicAdd(&s_cnt[C_RAY], (unsigned long long)(n_sc - n_hg));
      atomicAdd(&s_cnt[C_HG], (unsigned long long)n_hg);
      atomicAdd(&s_cnt[C_SFC_HITS], (unsigned long long)n_sfc);
      atomicAdd(&s_cnt[C_CELLS], (unsigned long long)n_cells);
      atomicAdd(&s_cnt[fate == 1 ? C_ATM_ABS : fate == 2 ? C_SFC_ABS : fate == 3 ? C_TOA : C_CAPPED], 1ull);
      if (fate == 4) atomicAdd(&s_cnt[C_CAPPED_E], kW0);
      if (kRecords) {
        uint4 r;
        r.x = (uint32_t)fate | (min(n_sfc, 0xFFFFFFu) << 8);
        r.y = term; r.z = n_ev; r.w = n_sc;
        reinterpret_cast<uint4*>(A.records)[i] = r;
      }
      alive = false;
    }
  }

  __syncthreads();
  if (threadIdx.x < C_COUNT && s_cnt[threadIdx.x] != 0ull)
    atomicAdd(&A.counters[threadIdx.x], s_cnt[threadIdx.x]);
}

}  // namespace rt
