// rt_setup.cuh — set-up kernels run by rt_set_optics and the random-gather
// microbenchmark behind rt_gather_bench.
#pragma once
#include "rt_device.cuh"

namespace rt {

// §3.4 pack cumulative coefficients; §3.5 majorant = highest extinction coefficient in each
// acceleration cell.  One thread per voxel, x fastest, so loads and the float4 store are
// coalesced.  Non-negative floats order like their bit patterns, so the cell maximum is an
// integer atomicMax (exact).  `bad` receives a bit mask of violated input ranges.
__global__ void pack_optics_kernel(const float* __restrict__ k_ext, const float* __restrict__ k_cloud,
                                   const float* __restrict__ ssa, const float* __restrict__ g,
                                   float4* __restrict__ optics, int* __restrict__ khat_bits,
                                   int* __restrict__ kmin_bits, int nx, int ny,
                                   int nz, int bx, int by, int bz, int* __restrict__ bad) {
  const size_t nvox = (size_t)nx * ny * nz;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  const int ncx = nx / bx, ncy = ny / by;
  for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < nvox; v += stride) {
    const float k = k_ext[v], kc = k_cloud[v], w = ssa[v], gg = g[v];
    int flags = 0;
    if (!(k >= 0.0f) || isinf(k)) flags |= 1;
    if (!(kc >= 0.0f) || !(kc <= k)) flags |= 2;
    if (!(w >= 0.0f) || !(w <= 1.0f)) flags |= 4;
    if (!(fabsf(gg) < 1.0f)) flags |= 8;
    if (flags) atomicOr(bad, flags);
    float c3 = k;
    float c1 = (1.0f - w) * k;
    const float frac = (k > 0.0f) ? kc / k : 0.0f;
    float c2 = c1 + (w * k) * frac;
    c2 = fminf(c2, c3);
    c1 = fminf(c1, c2);
    optics[v] = make_float4(c1, c2, c3, gg);
    const int x = (int)(v % nx), y = (int)((v / nx) % ny), z = (int)(v / ((size_t)nx * ny));
    const int cell = ((z / bz) * ncy + (y / by)) * ncx + (x / bx);
    // lanes of a warp that share a cell: reduce before the atomic
    const unsigned act = __activemask();
    const unsigned peers = __match_any_sync(act, cell);
    int m = flags ? 0 : __float_as_int(k);
    int mn = m;                              // §3.5b: the cell minimum, for the merge criterion
    const int leader = __ffs(peers) - 1;
    for (int off = 16; off > 0; off >>= 1) {
      const int o = __shfl_down_sync(act, m, off);
      const int on = __shfl_down_sync(act, mn, off);
      const unsigned src = (threadIdx.x & 31u) + off;
      if (src < 32u && ((peers >> src) & 1u)) { m = max(m, o); mn = min(mn, on); }
    }
    // shfl_down reduction is only complete when peers are contiguous; contiguous x runs are,
    // but guard the general case with a per-lane atomic when they are not.
    const unsigned run = peers >> leader;
    const bool contiguous = (run & (run + 1u)) == 0u;
    if (contiguous) {
      if ((int)(threadIdx.x & 31u) == leader) {
        atomicMax(&khat_bits[cell], m);
        if (kmin_bits) atomicMin(&kmin_bits[cell], mn);
      }
    } else {
      atomicMax(&khat_bits[cell], flags ? 0 : __float_as_int(k));
      if (kmin_bits) atomicMin(&kmin_bits[cell], flags ? 0 : __float_as_int(k));
    }
  }
}

// The same step for grids whose nx is a multiple of 4 (all of BASELINE.json's): one (z, y) row per block
// iteration, four consecutive voxels per thread: 16-byte loads of the four input fields, four 16-byte
// stores, no per-voxel index division; cell maximum (and minimum) reduced over the thread's voxels of the
// same cell before the atomics.  Streaming, HBM-bound: 32 B per voxel.
__device__ __forceinline__ float4 pack_one(float k, float kc, float w, float gg, int& flags) {
  if (!(k >= 0.0f) || isinf(k)) flags |= 1;
  if (!(kc >= 0.0f) || !(kc <= k)) flags |= 2;
  if (!(w >= 0.0f) || !(w <= 1.0f)) flags |= 4;
  if (!(fabsf(gg) < 1.0f)) flags |= 8;
  const float c3 = k;
  float c1 = (1.0f - w) * k;
  const float frac = (k > 0.0f) ? kc / k : 0.0f;
  float c2 = c1 + (w * k) * frac;
  c2 = fminf(c2, c3);
  c1 = fminf(c1, c2);
  return make_float4(c1, c2, c3, gg);
}

__global__ void __launch_bounds__(128) pack_optics_rows_kernel(
    const float4* __restrict__ k_ext, const float4* __restrict__ k_cloud, const float4* __restrict__ ssa,
    const float4* __restrict__ g, float4* __restrict__ optics, int* __restrict__ khat_bits,
    int* __restrict__ kmin_bits, int nx, int ny, int nz, int bx, int by, int bz, int* __restrict__ bad) {
  const int nrows = ny * nz, ncx = nx / bx, ncy = ny / by, nx4 = nx >> 2;
  int flags = 0;
  for (int row = blockIdx.x; row < nrows; row += gridDim.x) {
    const int z = row / ny, y = row - z * ny;
    const int cellrow = ((z / bz) * ncy + (y / by)) * ncx;
    const size_t base4 = (size_t)row * nx4;
    for (int q = threadIdx.x; q < nx4; q += blockDim.x) {
      const float4 K = __ldcs(k_ext + base4 + q), KC = __ldcs(k_cloud + base4 + q), W = __ldcs(ssa + base4 + q),
                   G = __ldcs(g + base4 + q);
      int f = 0;
      float4* out = optics + (base4 + q) * 4;
      out[0] = pack_one(K.x, KC.x, W.x, G.x, f);
      out[1] = pack_one(K.y, KC.y, W.y, G.y, f);
      out[2] = pack_one(K.z, KC.z, W.z, G.z, f);
      out[3] = pack_one(K.w, KC.w, W.w, G.w, f);
      flags |= f;
      if (f) continue;                         // rt_set_optics fails anyway; keep bad bits out of the tables
      const float kv[4] = {K.x, K.y, K.z, K.w};
      int cell = cellrow + (q * 4) / bx;
      int hi = __float_as_int(kv[0]), lo = hi;
#pragma unroll
      for (int j = 1; j < 4; ++j) {
        const int cj = cellrow + (q * 4 + j) / bx;
        const int b = __float_as_int(kv[j]);
        if (cj != cell) {
          atomicMax(&khat_bits[cell], hi);
          if (kmin_bits) atomicMin(&kmin_bits[cell], lo);
          cell = cj; hi = b; lo = b;
        } else {
          hi = max(hi, b); lo = min(lo, b);
        }
      }
      atomicMax(&khat_bits[cell], hi);
      if (kmin_bits) atomicMin(&kmin_bits[cell], lo);
    }
  }
  if (flags) atomicOr(bad, flags);
}

// The same step without atomics, for bx in {1, 2, 4} (and nx a multiple of 4): one block iteration handles a
// whole ROW OF CELLS, i.e. the by x bz voxel rows that make up the cells (cy, cz) for all cx; a thread owns four
// consecutive voxels in x (4 / bx cells) in every one of those rows, so it sees all voxels of its cells and
// writes their maximum (and minimum) with plain stores: no atomics, no table to zero beforehand.
__global__ void __launch_bounds__(128) pack_optics_cellrows_kernel(
    const float4* __restrict__ k_ext, const float4* __restrict__ k_cloud, const float4* __restrict__ ssa,
    const float4* __restrict__ g, float4* __restrict__ optics, float* __restrict__ khat, float* __restrict__ kmin,
    int nx, int ny, int nz, int bx, int by, int bz, int* __restrict__ bad) {
  const int ncx = nx / bx, ncy = ny / by, ncz = nz / bz, nx4 = nx >> 2;
  const int cells_per_thread = 4 / bx;               // 4, 2 or 1
  int flags = 0;
  for (int cr = blockIdx.x; cr < ncy * ncz; cr += gridDim.x) {
    const int cz = cr / ncy, cy = cr - cz * ncy;
    for (int q = threadIdx.x; q < nx4; q += blockDim.x) {
      float hi[4] = {0.0f, 0.0f, 0.0f, 0.0f};
      float lo[4] = {INFINITY, INFINITY, INFINITY, INFINITY};
      for (int dz_ = 0; dz_ < bz; ++dz_)
        for (int dy_ = 0; dy_ < by; ++dy_) {
          const size_t base4 = ((size_t)(cz * bz + dz_) * ny + (size_t)(cy * by + dy_)) * nx4 + q;
          const float4 K = __ldcs(k_ext + base4), KC = __ldcs(k_cloud + base4), W = __ldcs(ssa + base4),
                       G = __ldcs(g + base4);
          float4* out = optics + base4 * 4;
          out[0] = pack_one(K.x, KC.x, W.x, G.x, flags);
          out[1] = pack_one(K.y, KC.y, W.y, G.y, flags);
          out[2] = pack_one(K.z, KC.z, W.z, G.z, flags);
          out[3] = pack_one(K.w, KC.w, W.w, G.w, flags);
          hi[0] = fmaxf(hi[0], K.x); hi[1] = fmaxf(hi[1], K.y); hi[2] = fmaxf(hi[2], K.z); hi[3] = fmaxf(hi[3], K.w);
          lo[0] = fminf(lo[0], K.x); lo[1] = fminf(lo[1], K.y); lo[2] = fminf(lo[2], K.z); lo[3] = fminf(lo[3], K.w);
        }
      // per x position so far; now over the bx positions of each cell
      const size_t cell0 = ((size_t)cz * ncy + cy) * ncx + (size_t)q * cells_per_thread;
      if (bx == 1) {
#pragma unroll
        for (int j = 0; j < 4; ++j) { khat[cell0 + j] = hi[j]; if (kmin) kmin[cell0 + j] = lo[j]; }
      } else if (bx == 2) {
        khat[cell0] = fmaxf(hi[0], hi[1]); khat[cell0 + 1] = fmaxf(hi[2], hi[3]);
        if (kmin) { kmin[cell0] = fminf(lo[0], lo[1]); kmin[cell0 + 1] = fminf(lo[2], lo[3]); }
      } else {
        khat[cell0] = fmaxf(fmaxf(hi[0], hi[1]), fmaxf(hi[2], hi[3]));
        if (kmin) kmin[cell0] = fminf(fminf(lo[0], lo[1]), fminf(lo[2], lo[3]));
      }
    }
  }
  if (flags) atomicOr(bad, flags);
}

// Factored inputs (the optical properties of a spectral point are a gas part that
// depends on height only plus the cloud part): per voxel, in fp32 and in this order,
//   k_ext = (k_abs[z] + k_ray[z]) + k_cloud;  ssa = (k_ray[z] + cloud_ssa * k_cloud) / k_ext (0 if k_ext = 0);
//   g = cloud_g;  then the packing of §3.4.  Same cell-row scheme as above, reading 4 B per voxel instead of 16.
__global__ void __launch_bounds__(128) pack_factored_cellrows_kernel(
    const float4* __restrict__ k_cloud, const float* __restrict__ k_abs, const float* __restrict__ k_ray,
    float cloud_ssa, float cloud_g, float4* __restrict__ optics, float* __restrict__ khat, float* __restrict__ kmin,
    int nx, int ny, int nz, int bx, int by, int bz, int* __restrict__ bad) {
  const int ncx = nx / bx, ncy = ny / by, ncz = nz / bz, nx4 = nx >> 2;
  const int cells_per_thread = 4 / bx;
  int flags = 0;
  for (int cr = blockIdx.x; cr < ncy * ncz; cr += gridDim.x) {
    const int cz = cr / ncy, cy = cr - cz * ncy;
    for (int q = threadIdx.x; q < nx4; q += blockDim.x) {
      float hi[4] = {0.0f, 0.0f, 0.0f, 0.0f};
      float lo[4] = {INFINITY, INFINITY, INFINITY, INFINITY};
      for (int dz_ = 0; dz_ < bz; ++dz_) {
        const int z = cz * bz + dz_;
        const float ka = __ldg(k_abs + z), kr = __ldg(k_ray + z);
        const float kg = ka + kr;
        if (!(ka >= 0.0f) || !(kr >= 0.0f) || isinf(kg)) flags |= 1;
        for (int dy_ = 0; dy_ < by; ++dy_) {
          const size_t base4 = ((size_t)z * ny + (size_t)(cy * by + dy_)) * nx4 + q;
          const float4 KC = __ldcs(k_cloud + base4);
          const float kc[4] = {KC.x, KC.y, KC.z, KC.w};
          float4* out = optics + base4 * 4;
          float k[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            k[j] = kg + kc[j];
            const float w = (k[j] > 0.0f) ? (kr + cloud_ssa * kc[j]) / k[j] : 0.0f;
            out[j] = pack_one(k[j], kc[j], w, cloud_g, flags);
          }
          hi[0] = fmaxf(hi[0], k[0]); hi[1] = fmaxf(hi[1], k[1]); hi[2] = fmaxf(hi[2], k[2]); hi[3] = fmaxf(hi[3], k[3]);
          lo[0] = fminf(lo[0], k[0]); lo[1] = fminf(lo[1], k[1]); lo[2] = fminf(lo[2], k[2]); lo[3] = fminf(lo[3], k[3]);
        }
      }
      const size_t cell0 = ((size_t)cz * ncy + cy) * ncx + (size_t)q * cells_per_thread;
      if (bx == 1) {
#pragma unroll
        for (int j = 0; j < 4; ++j) { khat[cell0 + j] = hi[j]; if (kmin) kmin[cell0 + j] = lo[j]; }
      } else if (bx == 2) {
        khat[cell0] = fmaxf(hi[0], hi[1]); khat[cell0 + 1] = fmaxf(hi[2], hi[3]);
        if (kmin) { kmin[cell0] = fminf(lo[0], lo[1]); kmin[cell0 + 1] = fminf(lo[2], lo[3]); }
      } else {
        khat[cell0] = fmaxf(fmaxf(hi[0], hi[1]), fmaxf(hi[2], hi[3]));
        if (kmin) kmin[cell0] = fminf(fminf(lo[0], lo[1]), fminf(lo[2], lo[3]));
      }
    }
  }
  if (flags) atomicOr(bad, flags);
}

// Factored optics kept factored (rt_set_cloud + rt_set_point): the cloud field is stored once; what depends on the
// spectral point is built from small tables.  cloud_levels_kernel: per acceleration cell and per level inside the
// cell, the highest and lowest cloud extinction over the cell's bx x by voxels of that level ([cell][bz] floats).
// fl(gas[z] + k_cloud) is monotone in k_cloud, so the extrema of k_ext over the cell follow from these tables
// exactly (point_majorant_kernel), without touching the field again.
__global__ void cloud_levels_kernel(const float* __restrict__ k_cloud, float* __restrict__ cmax, float* __restrict__ cmin,
                                    int nx, int ny, int nz, int bx, int by, int bz, int* __restrict__ bad) {
  const int ncx = nx / bx, ncy = ny / by, ncz = nz / bz;
  const size_t n = (size_t)ncx * ncy * ncz * bz;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += stride) {
    // t = ((cz * bz + dz) * ncy + cy) * ncx + cx: consecutive threads read neighbouring x
    const int cx = (int)(t % ncx), cy = (int)((t / ncx) % ncy), z = (int)(t / ((size_t)ncx * ncy));
    float hi = 0.0f, lo = INFINITY;
    bool ok = true;
    for (int dy_ = 0; dy_ < by; ++dy_)
      for (int dx_ = 0; dx_ < bx; ++dx_) {
        const float k = k_cloud[((size_t)z * ny + (size_t)(cy * by + dy_)) * nx + (size_t)(cx * bx + dx_)];
        if (!(k >= 0.0f) || isinf(k)) ok = false;
        hi = fmaxf(hi, k); lo = fminf(lo, k);
      }
    if (!ok) atomicOr(bad, 2);
    const size_t cell = ((size_t)(z / bz) * ncy + cy) * ncx + cx;
    cmax[cell * bz + (z % bz)] = hi;
    cmin[cell * bz + (z % bz)] = lo;
  }
}

// Majorant (and per-cell minimum, for the merge criterion) of one spectral point from the cloud level tables and
// the point's gas profiles: k_hat[cell] = max over the cell's levels of fl((k_abs[z] + k_ray[z]) + cmax).
__global__ void point_majorant_kernel(const float* __restrict__ cmax, const float* __restrict__ cmin,
                                      const float* __restrict__ k_abs, const float* __restrict__ k_ray,
                                      float* __restrict__ khat, float* __restrict__ kmin, int ncx, int ncy, int ncz,
                                      int bz, int* __restrict__ bad) {
  const size_t ncell = (size_t)ncx * ncy * ncz;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < ncell; c += stride) {
    const int cz = (int)(c / ((size_t)ncx * ncy));
    float hi = 0.0f, lo = INFINITY;
    for (int dz_ = 0; dz_ < bz; ++dz_) {
      const float ka = __ldg(k_abs + cz * bz + dz_), kr = __ldg(k_ray + cz * bz + dz_);
      const float kg = ka + kr;
      if (!(ka >= 0.0f) || !(kr >= 0.0f) || isinf(kg)) atomicOr(bad, 1);
      hi = fmaxf(hi, kg + cmax[c * bz + dz_]);
      lo = fminf(lo, kg + cmin[c * bz + dz_]);
    }
    khat[c] = hi;
    if (kmin) kmin[c] = lo;
  }
}

// Voxel-sized cells with the optics kept factored: no majorant table per spectral point at all.  The level-0 majorant of
// a voxel is fl((k_abs[z] + k_ray[z]) + k_cloud), which MOVE computes from the shared cloud field; what remains per
// point is one word per BLOCK of mx x my x mz cells: -(block maximum) if the block is merged (§3.5b), else +maximum.
// cloud_blocks_kernel (once per cloud field): per block and per level inside it, the extrema of the cloud extinction
// ([block][mz * bz] floats); one warp per block.
__global__ void cloud_blocks_kernel(const float* __restrict__ k_cloud, float* __restrict__ bmax, float* __restrict__ bmin,
                                    int nx, int ny, int nz, int sx, int sy, int sz, int* __restrict__ bad) {
  const int nbx = nx / sx, nby = ny / sy, nbz = nz / sz;
  const size_t nblk = (size_t)nbx * nby * nbz;
  const size_t b = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (b >= nblk) return;
  const unsigned lane = threadIdx.x & 31u;
  const int X = (int)(b % nbx), Y = (int)((b / nbx) % nby), Z = (int)(b / ((size_t)nbx * nby));
  bool ok = true;
  for (int lz = 0; lz < sz; ++lz) {
    float hi = 0.0f, lo = INFINITY;
    for (int k = (int)lane; k < sx * sy; k += 32) {
      const int x = X * sx + k % sx, y = Y * sy + k / sx, z = Z * sz + lz;
      const float v = k_cloud[((size_t)z * ny + y) * nx + x];
      if (!(v >= 0.0f) || isinf(v)) ok = false;
      hi = fmaxf(hi, v); lo = fminf(lo, v);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, off));
      lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, off));
    }
    if (lane == 0) { bmax[b * sz + lz] = hi; bmin[b * sz + lz] = lo; }
  }
  if (!ok) atomicOr(bad, 2);
}

// point_blocks_kernel (blockIdx.y = spectral point p of the call): gsum[p][z] = fl(k_abs[z] + k_ray[z]) and the block
// words of the point.  fl(gsum + k_cloud) is monotone in k_cloud, so the block's extrema of k_ext follow exactly from
// the cloud extrema per level.  gas: the points' profiles as rt.cu keeps them (per point k_abs[nz] then k_ray[nz]).
__global__ void point_blocks_kernel(const float* __restrict__ bmax, const float* __restrict__ bmin,
                                    const float* __restrict__ gas, float* __restrict__ gsum, float* __restrict__ btab,
                                    int nbx, int nby, int nbz, int sz, int nz, float merge_ratio, int* __restrict__ bad) {
  const size_t nblk = (size_t)nbx * nby * nbz;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  const size_t pt = blockIdx.y;
  const float* k_abs = gas + pt * 2 * (size_t)nz;
  const float* k_ray = k_abs + nz;
  gsum += pt * (size_t)nz; btab += pt * nblk; bad += pt;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < (size_t)nz; t += stride) {
    const float ka = __ldg(k_abs + t), kr = __ldg(k_ray + t);
    const float kg = ka + kr;
    if (!(ka >= 0.0f) || !(kr >= 0.0f) || isinf(kg)) atomicOr(bad, 1);
    gsum[t] = kg;
  }
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < nblk; t += stride) {
    const int Z = (int)(t / ((size_t)nbx * nby));
    float hi = 0.0f, lo = INFINITY;
    for (int lz = 0; lz < sz; ++lz) {
      const float kg = __ldg(k_abs + Z * sz + lz) + __ldg(k_ray + Z * sz + lz);
      hi = fmaxf(hi, kg + bmax[t * sz + lz]);
      lo = fminf(lo, kg + bmin[t * sz + lz]);
    }
    btab[t] = (hi <= merge_ratio * lo) ? -hi : hi;
  }
}

// Albedo slots of several points at once (blockIdx.y = point of the call): range check into the point's mask word;
// broadcast != 0: every point takes the first slot's albedo (already copied there).
__global__ void albedo_points_kernel(float* __restrict__ albedo, size_t ncol, int broadcast, int* __restrict__ bad) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  const size_t pt = blockIdx.y;
  bool ok = true;
  for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < ncol; c += stride) {
    const float a = broadcast ? albedo[c] : albedo[pt * ncol + c];
    if (broadcast && pt > 0) albedo[pt * ncol + c] = a;
    if (!(a >= 0.0f) || !(a <= 1.0f)) ok = false;
  }
  if (!ok) atomicOr(bad + pt, 16);
}

// §3.5b merged cells.  One WARP per block of mx x my x mz acceleration cells (lanes stride over the block's
// cells, x fastest): if the block's highest extinction is at most merge_ratio times its lowest (one fp32
// multiply), every cell of the block stores -(block maximum); the sign bit is what the trace kernel tests
// (set also for a maximum of 0).
__global__ void merge_cells_kernel(float* __restrict__ khat, const float* __restrict__ kmin, int ncx, int ncy,
                                   int ncz, int mx, int my, int mz, float merge_ratio) {
  const int nbx = ncx / mx, nby = ncy / my, nbz = ncz / mz;
  const size_t nblk = (size_t)nbx * nby * nbz;
  const size_t b = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (b >= nblk) return;                             // whole warps leave together
  const unsigned lane = threadIdx.x & 31u;
  const int X = (int)(b % nbx), Y = (int)((b / nbx) % nby), Z = (int)(b / ((size_t)nbx * nby));
  const int ncell = mx * my * mz;
  float hi = 0.0f, lo = INFINITY;
  for (int k = (int)lane; k < ncell; k += 32) {
    const int x = X * mx + k % mx, y = Y * my + (k / mx) % my, z = Z * mz + k / (mx * my);
    const size_t c = ((size_t)z * ncy + y) * ncx + x;
    hi = fmaxf(hi, khat[c]);
    lo = fminf(lo, kmin[c]);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, off));
    lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, off));
  }
  if (!(hi <= merge_ratio * lo)) return;
  const float v = -hi;
  for (int k = (int)lane; k < ncell; k += 32) {
    const int x = X * mx + k % mx, y = Y * my + (k / mx) % my, z = Z * mz + k / (mx * my);
    khat[((size_t)z * ncy + y) * ncx + x] = v;
  }
}

__global__ void check_albedo_kernel(const float* __restrict__ albedo, size_t ncol, int* __restrict__ bad) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < ncol; c += stride) {
    const float a = albedo[c];
    if (!(a >= 0.0f) || !(a <= 1.0f)) atomicOr(bad, 16);
  }
}

// Random 16-byte gathers over the packed-optics array: 8 independent loads in flight per thread.
__global__ void gather_bench_kernel(const float4* __restrict__ optics, unsigned long long nvox,
                                    uint32_t iters, float* __restrict__ sink) {
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  float acc = 0.0f;
  for (uint32_t it = 0; it < iters; ++it) {
    const uint4 a = philox4x32_10(tid, it, 0u, 0x9a7e12u, 7u, 11u);
    const uint4 b = philox4x32_10(tid, it, 1u, 0x9a7e12u, 7u, 11u);
    const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
    float4 v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = __ldg(&optics[(size_t)(((unsigned long long)w[j] * nvox) >> 32)]);
#pragma unroll
    for (int j = 0; j < 8; ++j) acc += v[j].x + v[j].w;
  }
  if (acc == -1.2345f) sink[0] = acc;
}

// rt_selftest_ieee: rcp_in_range and sqrt_in_range (rt_device.cuh) against the IEEE operations they stand for, over
// EVERY float of their ranges: bit patterns [lo, hi) of positive floats, the reciprocal also for the negated value.
__global__ void ieee_selftest_kernel(unsigned long long* __restrict__ bad, uint32_t rcp_lo, uint32_t rcp_hi,
                                     uint32_t sqrt_lo, uint32_t sqrt_hi) {
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  const unsigned long long t0 = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long nr = 0, ns = 0;
  for (unsigned long long b = rcp_lo + t0; b < rcp_hi; b += stride) {
    const float x = __uint_as_float((uint32_t)b);
    if (__float_as_uint(rcp_in_range(x)) != __float_as_uint(1.0f / x)) ++nr;
    if (__float_as_uint(rcp_in_range(-x)) != __float_as_uint(1.0f / -x)) ++nr;
  }
  for (unsigned long long b = sqrt_lo + t0; b < sqrt_hi; b += stride) {
    const float x = __uint_as_float((uint32_t)b);
    if (__float_as_uint(sqrt_in_range(x)) != __float_as_uint(sqrtf(x))) ++ns;
  }
  if (nr) atomicAdd(bad, nr);
  if (ns) atomicAdd(bad + 1, ns);
}

__global__ void philox_words_kernel(const uint4* __restrict__ ctr, uint32_t k0, uint32_t k1,
                                    uint4* __restrict__ out, unsigned long long n) {
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
    const uint4 c = ctr[j];
    out[j] = philox4x32_10(c.x, c.y, c.z, c.w, k0, k1);
  }
}

}  // namespace rt
