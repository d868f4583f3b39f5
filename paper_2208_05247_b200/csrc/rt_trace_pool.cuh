// rt_trace_pool.cuh — the photon-tracing kernel organised around warp-private PHOTON POOLS in shared memory
// (same per-photon operation sequence as DESIGN.md §3.6-3.14, so the results are bit-identical
// to rt_trace.cuh's and to the oracle's kernel-precision instantiation).
//
// Why.  With one photon per lane (rt_trace.cuh) a warp can only run a phase for the lanes whose photon happens
// to need it: ncu showed 15 of 32 lanes active per issued instruction (profiles/r1b_trace_kernel.md), and a
// queueing argument bounds any vote-scheduled one-photon-per-lane kernel near 50 %.  Here a warp owns up to
// kPoolT photons, three to four times its lanes.  Their state (64 bytes, 80 with a weight / point / record
// counters) lives in shared memory in four stacks, one per phase the photon waits for:
//   M  MOVE      one step of the remaining-distance traversal (§3.7): cross a face or find the collision
//   C  COLLIDE   voxel gather, deposit / classification, draw of the next event (§3.8)
//   S  SCATTER   phase-function angle, rotation, new face distances (§3.9)
//   B  BOUNDARY  surface (§3.10), domain top (§3.11), change of level at a merged cell's face (§3.7b)
// Every iteration the warp picks a stack that holds at least 32 photons (priority S, C, B, M; else it launches
// 32 new photons, §3.6; partial batches only when nothing else is possible), pops the top 32 records with four
// conflict-free 16-byte shared-memory loads per lane, runs the phase with ALL lanes, and pushes each photon
// onto the stack of the phase it needs next (ballot + popcount give the compacted positions).  The stack sizes
// are warp-uniform scalars, so there is no vote, and no lane ever waits for a batch to fill.
//
// Layout per warp: planes[p][slot] of 16 bytes, slot-major inside a plane, so lane l reading slot s0 + l touches
// consecutive 16-byte words.  Slots [0, kPoolT): M grows up from 0, B grows down from kPoolT - 1 (M + B <= the
// photons the warp holds <= kPoolT).  Slots [kPoolT, kPoolT + kPoolCS): C grows up, S grows down; C + S <= 94
// because S runs at 32, C runs at 32 only when S < 32, and M (which feeds C) only when both are below 32.
#pragma once
#include "rt_trace.cuh"

namespace rt {

#ifndef RT_POOL_T
#define RT_POOL_T 96
#endif
#ifndef RT_POOL_WARPS
#define RT_POOL_WARPS 4
#endif
#ifndef RT_POOL_BLOCKS
#define RT_POOL_BLOCKS 4
#endif
#ifndef RT_POOL_MOVE_STEPS
#define RT_POOL_MOVE_STEPS 2
#endif
constexpr int kPoolT = RT_POOL_T;              // photons a warp holds at most (multiple of 32)
constexpr int kPoolCS = 96;                    // slots of the C/S region (>= 94, see above)
constexpr int kPoolSlots = kPoolT + kPoolCS;
constexpr int kPoolWarps = RT_POOL_WARPS;      // warps per block
constexpr int kPoolThreads = kPoolWarps * 32;
constexpr int kPoolBlocksPerSM = RT_POOL_BLOCKS;   // launch bound (registers); the resident count comes from the occupancy query
constexpr int kPoolMoveSteps = RT_POOL_MOVE_STEPS; // MOVE steps per visit of the M stack

__host__ __device__ constexpr int pool_planes(bool wide) { return wide ? 5 : 4; }
__host__ __device__ constexpr size_t pool_smem_bytes(bool wide) {
  return (size_t)kPoolWarps * pool_planes(wide) * kPoolSlots * 16;
}

// cell index packed in one word: cx, cy < 2048, -64 <= cz < 960 (rt_create_grid checks the grid against these)
constexpr int kCellBits = 11, kCellZBias = 64;
constexpr uint32_t kCellMask = (1u << kCellBits) - 1u;

enum : int { OUT_NONE = 0, OUT_M = 1, OUT_C = 2, OUT_S = 3, OUT_B = 4 };

template <bool kRecords, bool kPow2, bool kWeighted, bool kBatch>
__global__ void __launch_bounds__(kPoolThreads, kPoolBlocksPerSM) trace_pool_kernel(const TraceArgs A) {
  constexpr bool kWide = kRecords || kWeighted || kBatch;
  constexpr int kPlanes = pool_planes(kWide);
  extern __shared__ uint4 pool_smem[];
  __shared__ unsigned long long s_cnt[C_COUNT];
  if (threadIdx.x < C_COUNT) s_cnt[threadIdx.x] = 0ull;
  __syncthreads();

  const unsigned lane = threadIdx.x & 31u;
  const unsigned lt_mask = (1u << lane) - 1u;
  uint4* const pool = pool_smem + (size_t)(threadIdx.x >> 5) * kPlanes * kPoolSlots;

  // stack sizes (warp-uniform)
  int nM = 0, nB = 0, nC = 0, nS = 0;
  bool exhausted = false;

  // the photon this lane works on during a phase
  float rx, ry, rz, tau, delx, dely, delz, kh, da, db, dc;
  uint32_t pyz, cell, i, pzw, pe;
  uint32_t x0 = 0, x1 = 0, x2 = 0, x3 = 0;   // wide records: weight - 1, point, n_ev | n_sfc low << 21, n_sc | n_sfc high << 21

  // running totals of this thread (any photon it happened to process)
  uint32_t t_ev = 0, t_sc = 0, t_hg = 0, t_sfc = 0, t_cells = 0, t_relevel = 0, t_rkept = 0;
  unsigned long long t_rlost = 0, t_rgain = 0;

  auto pop = [&](int slot) {
    const uint4 a = pool[slot], b = pool[kPoolSlots + slot], c = pool[2 * kPoolSlots + slot], d = pool[3 * kPoolSlots + slot];
    rx = __uint_as_float(a.x); ry = __uint_as_float(a.y); rz = __uint_as_float(a.z); tau = __uint_as_float(a.w);
    delx = __uint_as_float(b.x); dely = __uint_as_float(b.y); delz = __uint_as_float(b.z); kh = __uint_as_float(b.w);
    da = __uint_as_float(c.x); db = __uint_as_float(c.y); dc = __uint_as_float(c.z); pyz = c.w;
    cell = d.x; i = d.y; pzw = d.z; pe = d.w;
    if (kWide) { const uint4 w = pool[4 * kPoolSlots + slot]; x0 = w.x; x1 = w.y; x2 = w.z; x3 = w.w; }
  };
  auto store = [&](int slot) {
    pool[slot] = make_uint4(__float_as_uint(rx), __float_as_uint(ry), __float_as_uint(rz), __float_as_uint(tau));
    pool[kPoolSlots + slot] = make_uint4(__float_as_uint(delx), __float_as_uint(dely), __float_as_uint(delz), __float_as_uint(kh));
    pool[2 * kPoolSlots + slot] = make_uint4(__float_as_uint(da), __float_as_uint(db), __float_as_uint(dc), pyz);
    pool[3 * kPoolSlots + slot] = make_uint4(cell, i, pzw, pe);
    if (kWide) pool[4 * kPoolSlots + slot] = make_uint4(x0, x1, x2, x3);
  };
  // push every lane's photon onto the stack `out` names; the masks are warp-uniform
  auto push = [&](int out) {
    const unsigned mM = __ballot_sync(0xffffffffu, out == OUT_M), mC = __ballot_sync(0xffffffffu, out == OUT_C);
    const unsigned mS = __ballot_sync(0xffffffffu, out == OUT_S), mB = __ballot_sync(0xffffffffu, out == OUT_B);
    int slot = nM + __popc(mM & lt_mask);
    if (out == OUT_B) slot = kPoolT - 1 - nB - __popc(mB & lt_mask);
    if (out == OUT_C) slot = kPoolT + nC + __popc(mC & lt_mask);
    if (out == OUT_S) slot = kPoolSlots - 1 - nS - __popc(mS & lt_mask);
    if (out != OUT_NONE) store(slot);
    nM += __popc(mM); nC += __popc(mC); nS += __popc(mS); nB += __popc(mB);
    __syncwarp();
  };

  // packed fields
  auto ev_index = [&]() { return pe & 0x1fffffu; };
  auto is_direct = [&]() { return (pe >> 21) & 1u; };
  auto y24 = [&]() { return pyz & 0xffffffu; };
  auto z24 = [&]() { return (pyz >> 24) | ((pzw & 0xffffu) << 8); };
  auto w24 = [&]() { return (pe >> 24) | ((pzw >> 16) << 8); };
  auto u_of = [](uint32_t w) { return (float)w * 5.9604644775390625e-8f; };   // §3.2 on the word's top 24 bits
  auto sid = [&]() { return kBatch ? x1 : A.stream_id; };
  auto photon_id = [&]() { return A.first_id + A.index_base + (unsigned long long)i; };
  // §3.7 draw for event e: optical depth, and the three 24-bit uniforms kept packed until they are needed
  auto draw = [&](uint32_t e, uint32_t direct, uint32_t axis) {
    const unsigned long long pid = photon_id();
    const uint4 X = philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), e, sid(), A.keys);
    tau = neg_log(1.0f - u24(X.x));
    const uint32_t y = X.y >> 8, z = X.z >> 8, w = X.w >> 8;
    pyz = y | (z << 24);
    pzw = (z >> 8) | ((w >> 8) << 16);
    pe = e | (direct << 21) | (axis << 22) | (w << 24);
  };
  auto local = [&](float d, float r, float L) {
    const float v = nudge(d);
    return fminf(L, fmaxf(0.0f, fmaf(-v, r, v > 0.0f ? L : 0.0f)));
  };
  // §3.7 place(q): reciprocals, face spacings and remaining distances from local coordinates at the level kh names
  auto place = [&](float qx, float qy, float qz) {
    const bool lev = __float_as_int(kh) < 0;
    const float va = nudge(da), vb = nudge(db), vc = nudge(dc);
    const float ia = 1.0f / va, ib = 1.0f / vb, ic = 1.0f / vc;
    const float Lx = lev ? A.Lx1 : A.Lx, Ly = lev ? A.Ly1 : A.Ly, Lz = lev ? A.Lz1 : A.Lz;
    delx = Lx * fabsf(ia); dely = Ly * fabsf(ib); delz = Lz * fabsf(ic);
    rx = ((va > 0.0f ? Lx : 0.0f) - qx) * ia;
    ry = ((vb > 0.0f ? Ly : 0.0f) - qy) * ib;
    rz = ((vc > 0.0f ? Lz : 0.0f) - qz) * ic;
  };
  auto cell_index = [&](int cx, int cy, int cz) {
    const unsigned c = ((unsigned)cz * (unsigned)A.ncy + (unsigned)cy) * (unsigned)A.ncx + (unsigned)cx;
    return kBatch ? c + x1 * A.ncell32 : c;
  };
  auto pack_cell = [](int cx, int cy, int cz) {
    return (uint32_t)cx | ((uint32_t)cy << kCellBits) | ((uint32_t)(cz + kCellZBias) << (2 * kCellBits));
  };
  // §3.14 roulette; returns true if the photon ended (fate 5)
  int fate = 0;
  uint32_t term = 0;
  unsigned long long wq = kW0;
  auto roulette = [&](uint32_t where) {
    if (wq >= kW0 / 2) return false;
    const unsigned long long pid = photon_id();
    const uint4 Y = philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), ev_index() | 0x80000000u, sid(), A.keys);
    if ((unsigned long long)Y.w < wq) { t_rgain += kW0 - wq; ++t_rkept; wq = kW0; return false; }
    t_rlost += wq; fate = 5; term = where;
    return true;
  };
  // per-photon counts of the record (wide records only)
  auto rec_add_ev = [&]() { if (kRecords) x2 += 1u; };
  auto rec_add_sc = [&]() { if (kRecords) x3 += 1u; };
  auto rec_add_sfc = [&]() {
    if (kRecords) {
      uint32_t s = (x2 >> 21) | ((x3 >> 21) << 11);
      s = min(s + 1u, 0x3fffffu);
      x2 = (x2 & 0x1fffffu) | ((s & 0x7ffu) << 21);
      x3 = (x3 & 0x1fffffu) | ((s >> 11) << 21);
    }
  };
  // finished photons: tallies already issued by the phase; count the fates per warp, write the records
  auto finish = [&](bool have) {
    if (__any_sync(0xffffffffu, have && fate != 0)) {
      const unsigned f1 = __ballot_sync(0xffffffffu, have && fate == 1), f2 = __ballot_sync(0xffffffffu, have && fate == 2);
      const unsigned f3 = __ballot_sync(0xffffffffu, have && fate == 3), f4 = __ballot_sync(0xffffffffu, have && fate == 4);
      if (kWeighted) {
        const unsigned f5 = __ballot_sync(0xffffffffu, have && fate == 5);
        if (lane == 0 && f5) atomicAdd(&s_cnt[C_ROUL_KILLED], (unsigned long long)__popc(f5));
        if (have && fate == 4) atomicAdd(&s_cnt[C_CAPPED_E], wq);
      }
      if (lane == 0) {
        if (f1) atomicAdd(&s_cnt[C_ATM_ABS], (unsigned long long)__popc(f1));
        if (f2) atomicAdd(&s_cnt[C_SFC_ABS], (unsigned long long)__popc(f2));
        if (f3) atomicAdd(&s_cnt[C_TOA], (unsigned long long)__popc(f3));
        if (f4) {
          atomicAdd(&s_cnt[C_CAPPED], (unsigned long long)__popc(f4));
          if (!kWeighted) atomicAdd(&s_cnt[C_CAPPED_E], kW0 * (unsigned long long)__popc(f4));
        }
      }
      if (kRecords && have && fate != 0) {
        const uint32_t nsfc = (x2 >> 21) | ((x3 >> 21) << 11);
        uint4 r;
        r.x = (uint32_t)fate | (nsfc << 8);
        r.y = term; r.z = x2 & 0x1fffffu; r.w = x3 & 0x1fffffu;
        unsigned long long at = i;
        if (kBatch) at += __ldg(A.offsets + (x1 - (uint32_t)A.first_point));
        reinterpret_cast<uint4*>(A.records)[at] = r;
      }
    }
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
    t_ev = t_sc = t_hg = t_sfc = t_cells = t_relevel = t_rkept = 0;
    t_rlost = t_rgain = 0;
  };

  for (;;) {
    // ---- which phase: a stack with a full batch, else new photons, else the fullest stack ----------------
    int phase, n = 32;
    if (nS >= 32) phase = OUT_S;
    else if (nC >= 32) phase = OUT_C;
    else if (nB >= 32) phase = OUT_B;
    else if (nM >= 32) phase = OUT_M;
    else if (!exhausted && nM + nB + nC + nS + 32 <= kPoolT) phase = OUT_NONE;   // launch
    else {
      phase = OUT_S; n = nS;
      if (nC > n) { phase = OUT_C; n = nC; }
      if (nB > n) { phase = OUT_B; n = nB; }
      if (nM > n) { phase = OUT_M; n = nM; }
      if (n == 0) { if (exhausted) break; phase = OUT_NONE; }
    }
    const bool have = (int)lane < n;

    if (phase == OUT_NONE) {
      // ---- §3.6 launch, event index 0: 32 photon indices from the global counter -------------------------
      unsigned long long base = 0;
      if (lane == 0) base = atomicAdd(A.next_photon, 32ull);
      base = __shfl_sync(0xffffffffu, base, 0);
      if (base >= A.n_photons) { exhausted = true; continue; }
      if (__any_sync(0xffffffffu, t_ev > (1u << 30) || t_cells > (1u << 30))) flush_thread_counters();   // 32-bit totals
      const bool mine = base + lane < A.n_photons;
      int out = OUT_NONE;
      if (mine) {
        unsigned long long ii = base + lane;          // index in the launch
        unsigned long long n_full = A.n_full;
        x0 = x1 = x2 = x3 = 0;
        if (kBatch) {
          int lo = 0, hi = A.n_points;
          while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(A.offsets + mid) <= ii) lo = mid; else hi = mid;
          }
          x1 = (uint32_t)(lo + A.first_point);
          ii -= __ldg(A.offsets + lo);
          n_full = __ldg(A.nfull + lo);
        }
        i = (uint32_t)ii;
        const unsigned long long ij = A.index_base + ii;   // index in the job (the call): column and pass
        const unsigned long long pid = A.first_id + ij;
        const uint4 X = philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), 0u, sid(), A.keys);
        int ix, iy;
        float e0 = u24(X.x), e1 = u24(X.y);   // sub-pixel entry point
        if (ij < n_full) {
          const uint32_t col = (ij >> 32) ? (uint32_t)(ij % A.ncol) : (uint32_t)ij % (uint32_t)A.ncol;
          ix = (int)(col % (uint32_t)A.nx);
          iy = (int)(col / (uint32_t)A.nx);
          if (A.sobol) {
            const uint32_t k = (ij >> 32) ? (uint32_t)(ij / A.ncol) : (uint32_t)ij / (uint32_t)A.ncol;
            const uint4 S = philox4x32_10(col, sid(), (uint32_t)A.first_id, (uint32_t)(A.first_id >> 32), A.keys_sobol);
            uint32_t s1 = __brev(k), s2 = 0, V = 0x80000000u;
            for (uint32_t kk = k; kk; kk >>= 1) { if (kk & 1u) s2 ^= V; V ^= V >> 1; }
            e0 = u24(s1 ^ S.x); e1 = u24(s2 ^ S.y);
          }
        } else {
          ix = min((int)(u24(X.z) * (float)A.nx), A.nx - 1);
          iy = min((int)(u24(X.w) * (float)A.ny), A.ny - 1);
        }
        int cx = ix / A.bx, cy = iy / A.by, cz = A.ncz - 1;
        da = A.sun_x; db = A.sun_y; dc = A.sun_z;
        kh = __ldg(A.khat + cell_index(cx, cy, cz));
        const bool lev = __float_as_int(kh) < 0;
        int wx = A.bx, wy = A.by;
        float Lx = A.Lx, Ly = A.Ly, Lz = A.Lz;
        if (lev) {
          cx &= -A.mx; cy &= -A.my; cz &= -A.mz;
          wx *= A.mx; wy *= A.my; Lx = A.Lx1; Ly = A.Ly1; Lz = A.Lz1;
        }
        cell = pack_cell(cx, cy, cz);
        const float qx = ((float)(ix % wx) + e0) * A.dx, qy = ((float)(iy % wy) + e1) * A.dy;
        uint32_t direct = 1u;
        if (A.diffuse_fraction > 0.0f) {
          const uint4 D = philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), 0x80000000u, sid(), A.keys);
          if (u24(D.x) < A.diffuse_fraction) {
            const float v1 = u24(D.y);
            const float mu = sqrtf(1.0f - v1), sn = sqrtf(v1);
            float sp, cp;
            sincos_2pi(u24(D.z), sp, cp);
            da = sn * cp; db = sn * sp; dc = -mu;
            direct = 0u;
          }
        }
        if (direct) {
          delx = Lx * fabsf(A.sun_ix); dely = Ly * fabsf(A.sun_iy); delz = Lz * fabsf(A.sun_iz);
          rx = ((A.sun_ix > 0.0f ? Lx : 0.0f) - qx) * A.sun_ix;
          ry = ((A.sun_iy > 0.0f ? Ly : 0.0f) - qy) * A.sun_iy;
          rz = ((A.sun_iz > 0.0f ? Lz : 0.0f) - Lz) * A.sun_iz;
        } else {
          place(qx, qy, Lz);
        }
        if (kWeighted) x0 = 0xffffffffu;      // weight W0, stored as w - 1
        draw(1u, direct, 0u);
        out = OUT_M;
      }
      push(out);
      continue;
    }

    if (phase == OUT_M) {
      // ---- MOVE: nearest face of the current cell (ties x < y < z), then cross or stop (§3.7) ---------------
      int out = OUT_NONE;
      if (have) pop(nM - n + (int)lane);
      nM -= n;
      __syncwarp();
      if (have) {
        out = OUT_M;
        int cx = (int)(cell & kCellMask), cy = (int)((cell >> kCellBits) & kCellMask), cz = (int)(cell >> (2 * kCellBits)) - kCellZBias;
        const bool lev = __float_as_int(kh) < 0;
        const int sx = (da > -kTiny) ? (lev ? A.mx : 1) : (lev ? -A.mx : -1);
        const int sy = (db > -kTiny) ? (lev ? A.my : 1) : (lev ? -A.my : -1);
        const int sz = (dc > -kTiny) ? (lev ? A.mz : 1) : (lev ? -A.mz : -1);
#pragma unroll
        for (int rep = 0; rep < kPoolMoveSteps; ++rep) {
          if (out == OUT_M) {
            const bool ax0 = (rx <= ry) && (rx <= rz);
            const bool ax1 = !ax0 && (ry <= rz);
            const bool ax2 = !ax0 && !ax1;
            const float t = ax0 ? rx : (ax1 ? ry : rz);
            const float dtau = fabsf(kh) * t;
            if (fabsf(kh) > 0.0f && tau <= dtau) {
              out = OUT_C;                             // the tentative collision comes first
            } else {
              tau = tau - dtau;
              ++t_cells;
              rx = ax0 ? delx : rx - t;
              ry = ax1 ? dely : ry - t;
              rz = ax2 ? delz : rz - t;
              if (kPow2) {
                if (ax0) cx = (cx + sx) & (A.ncx - 1);
                if (ax1) cy = (cy + sy) & (A.ncy - 1);
              } else {
                if (ax0) { cx += sx; cx = (cx >= A.ncx) ? cx - A.ncx : cx; cx = (cx < 0) ? cx + A.ncx : cx; }
                if (ax1) { cy += sy; cy = (cy >= A.ncy) ? cy - A.ncy : cy; cy = (cy < 0) ? cy + A.ncy : cy; }
              }
              if (ax2) cz += sz;
              if ((unsigned)cz >= (unsigned)A.ncz) out = OUT_B;     // surface (cz < 0) or domain top
              else {
                const float raw = __ldg(A.khat + cell_index(cx, cy, cz));
                if ((__float_as_int(raw) ^ __float_as_int(kh)) < 0) {   // §3.7b: the entered cell is at the other level
                  out = OUT_B;
                  pe = (pe & ~(3u << 22)) | ((ax0 ? 0u : (ax1 ? 1u : 2u)) << 22);
                }
                kh = raw;
              }
            }
          }
        }
        cell = pack_cell(cx, cy, cz);
      }
      push(out);
      continue;
    }

    if (phase == OUT_S) {
      // ---- SCATTER: phase-function angle, rotation, new distances to the faces (§3.9) --------------------
      // S records hold (sg, word 2, word 3 of the scattering event) where M records hold the face spacings
      int out = OUT_NONE;
      if (have) pop(kPoolSlots - nS + (int)lane);
      nS -= n;
      __syncwarp();
      if (have) {
        const float sg = delx;
        const uint32_t sw2 = __float_as_uint(dely), sw3 = __float_as_uint(delz);
        const bool lev = __float_as_int(kh) < 0;
        const float qx = local(da, rx, lev ? A.Lx1 : A.Lx), qy = local(db, ry, lev ? A.Ly1 : A.Ly),
                    qz = local(dc, rz, lev ? A.Lz1 : A.Lz);
        float mu;
        if (sg < 1.5f) { mu = sample_hg(sg, u_of(sw2)); ++t_hg; }
        else           { mu = sample_rayleigh(u_of(sw2)); }
        float sp, cp;
        sincos_2pi(u_of(sw3), sp, cp);
        rotate_dir(da, db, dc, mu, cp, sp);
        place(qx, qy, qz);
        pe &= ~(1u << 21);                              // diffuse from now on
        ++t_sc; rec_add_sc();
        out = OUT_M;
      }
      push(out);
      continue;
    }

    fate = 0;
    term = 0;
    unsigned long long* tally_a = nullptr;  // arrival / terminal bin
    unsigned long long* tally_b = nullptr;  // surface absorption after an arrival tally
    int out = OUT_NONE;
    if (phase == OUT_C) {
      // ---- COLLIDE: fetch the voxel, classify, draw the next event (§3.8) ------------------------------
      if (have) pop(kPoolT + nC - n + (int)lane);
      nC -= n;
      __syncwarp();
      if (have) {
        if (kWeighted) wq = (unsigned long long)x0 + 1ull;
        const int cx = (int)(cell & kCellMask), cy = (int)((cell >> kCellBits) & kCellMask), cz = (int)(cell >> (2 * kCellBits)) - kCellZBias;
        const bool lev = __float_as_int(kh) < 0;
        const float rk = 1.0f / fabsf(kh);
        const float s = tau * rk;
        rx = fmaxf(0.0f, rx - s); ry = fmaxf(0.0f, ry - s); rz = fmaxf(0.0f, rz - s);
        const float qx = local(da, rx, lev ? A.Lx1 : A.Lx), qy = local(db, ry, lev ? A.Ly1 : A.Ly),
                    qz = local(dc, rz, lev ? A.Lz1 : A.Lz);
        const int lx = min((int)(qx * A.rdx), (lev ? A.mx * A.bx : A.bx) - 1);
        const int ly = min((int)(qy * A.rdy), (lev ? A.my * A.by : A.by) - 1);
        const int lz = min((int)(qz * A.rdz), (lev ? A.mz * A.bz : A.bz) - 1);
        const unsigned vox = ((unsigned)(cz * A.bz + lz) * (unsigned)A.ny + (unsigned)(cy * A.by + ly)) * (unsigned)A.nx
                             + (unsigned)(cx * A.bx + lx);
        float4 v;
        if (kBatch && A.cloud) {
          const float kc = __ldg(A.cloud + vox);
          const int z = cz * A.bz + lz;
          const float ka = __ldg(A.gas + (size_t)x1 * 2u * (unsigned)A.nz + z);
          const float kr = __ldg(A.gas + (size_t)x1 * 2u * (unsigned)A.nz + (unsigned)A.nz + z);
          const float2 pp = __ldg(A.point_par + x1);
          const float k = (ka + kr) + kc;                                     // §3.4b
          const float w = (k > 0.0f) ? (kr + pp.x * kc) / k : 0.0f;
          float c1 = (1.0f - w) * k;                                          // §3.4
          const float frac = (k > 0.0f) ? kc / k : 0.0f;
          float c2 = c1 + (w * k) * frac;
          c2 = fminf(c2, k);
          c1 = fminf(c1, c2);
          v = make_float4(c1, c2, k, pp.y);
        } else {
          v = __ldg(&A.optics[kBatch ? vox + x1 * A.nvox32 : vox]);
        }
        // the next event's draw does not depend on the voxel: issue it under the gather's latency
        const uint32_t e = ev_index(), direct = is_direct();
        const float u1 = u_of(y24());
        const uint32_t sw2 = z24(), sw3 = w24();          // this event's words 2, 3 (for a scatter)
        const float akh = fabsf(kh);
        draw(e + 1u, direct, 0u);                          // pe now names event e + 1
        ++t_ev; rec_add_ev();
        float xi = u1 * akh;
        out = OUT_M;
        if (kWeighted) {
          const float f = v.x * rk;
          const unsigned long long pq = min(1u << 24, (unsigned)(f * 16777216.0f));
          const unsigned long long a = (wq * pq) >> 24;
          if (a) atomicAdd(A.atm_abs + vox, a);
          if (a && direct && A.atm_dir) atomicAdd(A.atm_dir + vox, a);
          wq -= a;
          if (wq == 0) { fate = 1; term = (uint32_t)vox; }
          xi = fmaf(u1, akh - v.x, v.x);
        } else if (xi < v.x) {
          tally_a = A.atm_abs + vox;
          if (direct && A.atm_dir) atomicAdd(A.atm_dir + vox, kW0);
          fate = 1; term = (uint32_t)vox;
        }
        if (fate == 0) {
          bool scat = false;
          float sg = 0.0f;
          if (xi < v.z) { scat = true; sg = (xi < v.y) ? v.w : 2.0f; }
          bool ended = false;
          if (kWeighted) {
            // the roulette draws on the event's own counter: pe already names e + 1, so put e back for it
            const uint32_t pe_next = pe;
            pe = (pe & ~0x1fffffu) | e;
            ended = roulette((uint32_t)vox);
            pe = pe_next;
          }
          if (!ended && e + 1u > kEventCap) { fate = 4; term = 0; ended = true; }   // §3.12
          if (ended) {
            if (scat) { ++t_sc; rec_add_sc(); if (sg < 1.5f) ++t_hg; }             // the event itself is still counted
          } else if (scat) {
            out = OUT_S;
            delx = sg; dely = __uint_as_float(sw2); delz = __uint_as_float(sw3);
          }
        }
        if (fate != 0) out = OUT_NONE;
        if (kWeighted) x0 = (uint32_t)(wq - 1ull);
      }
    } else {
      // ---- BOUNDARY: change of level at a merged cell's face (§3.7b), surface (§3.10), domain top (§3.11) ---
      if (have) pop(kPoolT - nB + (int)lane);
      nB -= n;
      __syncwarp();
      if (have) {
        if (kWeighted) wq = (unsigned long long)x0 + 1ull;
        int cx = (int)(cell & kCellMask), cy = (int)((cell >> kCellBits) & kCellMask), cz = (int)(cell >> (2 * kCellBits)) - kCellZBias;
        out = OUT_M;
        if ((unsigned)cz < (unsigned)A.ncz) {
          const bool px = da > -kTiny, py = db > -kTiny, pz = dc > -kTiny;
          const int ax = (int)((pe >> 22) & 3u);
          const bool lev = !(__float_as_int(kh) < 0);   // kh already holds the ENTERED cell's word
          if (!lev) {
            const int ox = cx & (A.mx - 1), oy = cy & (A.my - 1), oz = cz & (A.mz - 1);
            const float fx = (float)A.mx, fy = (float)A.my, fz = (float)A.mz;
            rx = (ax == 0) ? delx * fx : fmaf((float)(px ? A.mx - 1 - ox : ox), delx, rx);
            ry = (ax == 1) ? dely * fy : fmaf((float)(py ? A.my - 1 - oy : oy), dely, ry);
            rz = (ax == 2) ? delz * fz : fmaf((float)(pz ? A.mz - 1 - oz : oz), delz, rz);
            delx *= fx; dely *= fy; delz *= fz;
            cx -= ox; cy -= oy; cz -= oz;
          } else {
            delx *= A.rmx; dely *= A.rmy; delz *= A.rmz;
            if (ax == 0) { rx = delx; if (!px) cx += A.mx - 1; }
            else { const int k = min(A.mx - 1, (int)(rx / delx)); rx = fmaxf(0.0f, fmaf(-(float)k, delx, rx)); cx += px ? A.mx - 1 - k : k; }
            if (ax == 1) { ry = dely; if (!py) cy += A.my - 1; }
            else { const int k = min(A.my - 1, (int)(ry / dely)); ry = fmaxf(0.0f, fmaf(-(float)k, dely, ry)); cy += py ? A.my - 1 - k : k; }
            if (ax == 2) { rz = delz; if (!pz) cz += A.mz - 1; }
            else { const int k = min(A.mz - 1, (int)(rz / delz)); rz = fmaxf(0.0f, fmaf(-(float)k, delz, rz)); cz += pz ? A.mz - 1 - k : k; }
            kh = __ldg(A.khat + cell_index(cx, cy, cz));
          }
          ++t_relevel;
          cell = pack_cell(cx, cy, cz);
        } else {
          const bool lev = __float_as_int(kh) < 0;
          const float qx = local(da, rx, lev ? A.Lx1 : A.Lx), qy = local(db, ry, lev ? A.Ly1 : A.Ly);
          const int hx = cx * A.bx + min((int)(qx * A.rdx), (lev ? A.mx * A.bx : A.bx) - 1);
          const int hy = cy * A.by + min((int)(qy * A.rdy), (lev ? A.my * A.by : A.by) - 1);
          const unsigned col = (unsigned)hy * (unsigned)A.nx + (unsigned)hx;
          const uint32_t direct = is_direct();
          if (cz >= 0) {
            if (kWeighted) atomicAdd(A.toa_up + col, wq); else tally_a = A.toa_up + col;
            fate = 3; term = (uint32_t)col;
          } else {
            ++t_sfc; rec_add_sfc();
            bool reflect;
            if (kWeighted) {
              atomicAdd((direct ? A.sfc_dir : A.sfc_dif) + col, wq);
              const unsigned long long aq = min(1u << 24, (unsigned)(__ldg(&A.albedo[kBatch ? col + x1 * A.ncol32 : col]) * 16777216.0f));
              const unsigned long long refl = (wq * aq) >> 24;
              if (wq - refl) atomicAdd(A.sfc_abs + col, wq - refl);
              wq = refl;
              if (wq == 0) { fate = 2; term = (uint32_t)col; reflect = false; }
              else reflect = !roulette((uint32_t)col);
            } else {
              tally_a = (direct ? A.sfc_dir : A.sfc_dif) + col;
              reflect = u_of(y24()) < __ldg(&A.albedo[kBatch ? col + x1 * A.ncol32 : col]);
              if (!reflect) { tally_b = A.sfc_abs + col; fate = 2; term = (uint32_t)col; }
            }
            if (reflect) {
              const float u2 = u_of(z24());
              const float mu = sqrtf(1.0f - u2), sn = sqrtf(u2);
              float sp, cp;
              sincos_2pi(u_of(w24()), sp, cp);
              da = sn * cp; db = sn * sp; dc = mu;
              cz = 0;                                   // back in the cell it left: same level, same majorant
              cell = pack_cell(cx, cy, cz);
              place(qx, qy, 0.0f);
              const uint32_t e = ev_index() + 1u;
              if (e > kEventCap) { fate = 4; term = 0; }   // §3.12
              else draw(e, 0u, 0u);
            }
          }
        }
        if (fate != 0) out = OUT_NONE;
        if (kWeighted) x0 = (uint32_t)(wq - 1ull);
      }
    }

    // ---- tallies: warp-aggregated 64-bit integer atomics ------------------------------------------------
    const unsigned ma = __ballot_sync(0xffffffffu, tally_a != nullptr);
    if (ma) {
      if (tally_a) tally_add(ma, tally_a);
      const unsigned mb = __ballot_sync(0xffffffffu, tally_b != nullptr);
      if (mb && tally_b) tally_add(mb, tally_b);
    }
    finish(have);
    push(out);
  }

  flush_thread_counters();
  __syncthreads();
  if (threadIdx.x == 0) s_cnt[C_NULL] -= s_cnt[C_ATM_ABS];   // events - scatters - absorptions
  __syncthreads();
  if (threadIdx.x < C_COUNT && s_cnt[threadIdx.x] != 0ull)
    atomicAdd(&A.counters[threadIdx.x], s_cnt[threadIdx.x]);
}

}  // namespace rt
