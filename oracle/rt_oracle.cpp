// rt_oracle.cpp — CPU ORACLE for the forward Monte Carlo shortwave photon tracer.
//
// TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may build, load or call this
// file.  The CUDA path (paper_2208_05247_b200/csrc) shares no code with it and
// never calls it; the two were written separately from the normative text in
// DESIGN.md §3 ("Stream definition").
//
// What it computes (§2.3 "The ray tracer"):
// photons launched at the domain top along the sun beam, propagated by
// single-level null-collision tracking on a coarse acceleration grid whose cell
// value is the highest extinction coefficient inside the cell, local
// optical properties fetched from the fine grid, Rayleigh / Henyey-
// Greenstein scattering chosen with probability k_ext,cloud/k_ext,
// Lambertian surface with local albedo, tallies of surface and
// domain-top fluxes and 3D absorbed power.  By default absorption is ANALOG
// (BASELINE.json north_star, reading D1): a photon ends in exactly one bin and
// carries W0 = 2^32 integer quanta, so energy closes exactly in int64.
// Options, each off by default and each with its own pins in tests/:
//   merged acceleration cells (tests/test_oracle_merged_cells.py),
//   the paper's absorption weights + Russian roulette (
//     tests/test_oracle_weighted.py), with the direct part of the heating,
//   the paper's top-of-domain source: scrambled Sobol entry points and a diffuse
//     fraction (tests/test_oracle_source.py).
//
// Plain, slow, single-threaded by definition (n_threads > 1 only splits the
// photon-id range for wall-clock timing; integer tallies make the result
// identical).  It follows DESIGN.md §3 step by step, in that order and
// notation, with no blocking, fusion or reordering.
//
// Precision.  The tracer is a template on Real:
//   Real = double : the oracle proper.  fp64 geometry, libm log/sin/cos/cbrt-
//                   free Rayleigh inversion.  Pinned by tests/test_oracle_*.py
//                   (Beer-Lambert, closure, limits, symmetry, single scatter,
//                   Philox known answers, sampler moments).
//   Real = float  : the same statements in the kernel's precision.  Every
//                   geometric comparison decides an integer (which cell face,
//                   which voxel, which event), so for the per-photon identity
//                   criterion both sides take those decisions in fp32, using
//                   the fp32 elementary functions that DESIGN.md §3.3 fixes
//                   operation by operation (log, sincospi).  Every operation is
//                   an IEEE-754 correctly rounded +,-,*,/,sqrt,fma, so this
//                   instantiation is bit-reproducible on any conforming machine.
// Build with -ffp-contract=off (no implicit FMA); fma is written explicitly.
//
// Independent witness of the traversal and level-change arithmetic: tests/reference_walk.py (global
// coordinates, no levels, pure Python) must give the same photons, record by record.
// Parity unpinned: nothing.  (The cloud-vs-gas choice of P:56, "unpinned" in round 1, is pinned by
// tests/test_oracle_split_cap_precision.py against the ratio the paper states; whether that ratio is the
// physically right one is the paper's own approximation, Q4 in DESIGN.md §2.)

#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>
#include <algorithm>
#include <chrono>

namespace {

// ---------------------------------------------------------------------------
// §3.1 Philox4x32-10 (Salmon et al., SC'11).  Constants as in the CUDA toolkit
// header curand_philox4x32_x.h (PHILOX_W32_0/1, PHILOX_M4x32_0/1).
// ---------------------------------------------------------------------------
struct U4 { uint32_t x, y, z, w; };

inline U4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                        uint32_t k0, uint32_t k1) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)M0 * c0;
    uint64_t p1 = (uint64_t)M1 * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  return U4{c0, c1, c2, c3};
}

// §3.2 word -> uniform in [0,1): top 24 bits, exact in fp32 and fp64.
template <class R> inline R uni24(uint32_t x) { return (R)(x >> 8) * (R)(1.0 / 16777216.0); }

// ---------------------------------------------------------------------------
// §3.3 fp32 elementary functions fixed operation by operation.
// ---------------------------------------------------------------------------
inline float spec_neg_log(float w) {  // -ln(w), w in [2^-24, 1]
  int32_t ix; std::memcpy(&ix, &w, 4);
  int32_t E = (ix - 0x3f3504f3) >> 23;         // arithmetic shift (floor)
  int32_t im = ix - (E << 23);
  float m; std::memcpy(&m, &im, 4);            // m in [sqrt(1/2), sqrt(2))
  float f = m - 1.0f;
  float P = 0x1.645de2p-4f;                    // Horner, degree 6 in f
  P = std::fmaf(P, f, -0x1.2432aap-3f);
  P = std::fmaf(P, f, 0x1.317470p-3f);
  P = std::fmaf(P, f, -0x1.53824cp-3f);
  P = std::fmaf(P, f, 0x1.98d7f0p-3f);
  P = std::fmaf(P, f, -0x1.000382p-2f);
  P = std::fmaf(P, f, 0x1.5556d8p-2f);
  float f2 = f * f;
  float r = std::fmaf(f * f2, P, -0.5f * f2);
  float l1p = f + r;
  float Ef = (float)E;
  float res = std::fmaf(Ef, 0x1.62e4p-1f, std::fmaf(Ef, 0x1.7f7d1cp-20f, l1p));
  return -res;
}

inline void spec_sincos_2pi(float u, float& sn_out, float& cs_out) {  // angle 2*pi*u, u in [0,1)
  float t = 2.0f * u;
  int j = (int)std::fmaf(2.0f, t, 0.5f);       // nearest quarter turn, 0..4
  float r = t - 0.5f * (float)j;               // exact, in [-1/4, 1/4]
  float z = r * r;
  float S = -0x1.2d9302p-1f;
  S = std::fmaf(S, z, 0x1.465e92p+1f);
  S = std::fmaf(S, z, -0x1.4abbbap+2f);
  S = std::fmaf(S, z, 0x1.921fb6p+1f);
  float sn = r * S;
  float C = 0x1.d99f54p-3f;
  C = std::fmaf(C, z, -0x1.55c4eap+0f);
  C = std::fmaf(C, z, 0x1.03c1dap+2f);
  C = std::fmaf(C, z, -0x1.3bd3ccp+2f);
  float cs = std::fmaf(C, z, 1.0f);
  switch (j & 3) {
    case 0: sn_out = sn;  cs_out = cs;  break;
    case 1: sn_out = cs;  cs_out = -sn; break;
    case 2: sn_out = -sn; cs_out = -cs; break;
    default: sn_out = -cs; cs_out = sn; break;
  }
}

// Real-generic wrappers: double uses the plain library definition.
template <class R> struct Elem;
template <> struct Elem<float> {
  static float neg_log_1m(float u) { return spec_neg_log(1.0f - u); }
  static void sincos_2pi(float u, float& s, float& c) { spec_sincos_2pi(u, s, c); }
  static float fma(float a, float b, float c) { return std::fmaf(a, b, c); }
};
template <> struct Elem<double> {
  static double neg_log_1m(double u) { return -std::log(1.0 - u); }
  static void sincos_2pi(double u, double& s, double& c) {
    const double two_pi = 6.283185307179586476925286766559;
    s = std::sin(two_pi * u); c = std::cos(two_pi * u);
  }
  static double fma(double a, double b, double c) { return std::fma(a, b, c); }
};

// ---------------------------------------------------------------------------
// §3.9 samplers
// ---------------------------------------------------------------------------
// Henyey-Greenstein ("Henyey-Greenstein phase function without delta-scaling"):
// inverse CDF of p(mu) = (1-g^2) / (2 (1 + g^2 - 2 g mu)^(3/2)), i.e. mu = (1 + g^2 - q^2) / (2 g) with
// q = (1 - g^2) / (1 - g + 2 g u).  Written in the cancellation-free form of DESIGN.md 3.9: with den = 1 - g + 2 g u,
//   1 - mu = (1 - g)(1 - u)(q + 1 - g) / den,     1 + mu = (1 + g) u (q + 1 + g) / den
// (their sum is 2 identically), mu = half their difference and sin(theta) = sqrt of their product, so the sine of
// a forward-peak angle keeps its relative accuracy in fp32 (1 - u is exact for a 24-bit u).  Regular at g = 0.
template <class R> inline void sample_hg(R g, R u, R& mu, R& s) {
  const R a = (R)1 - g, b = (R)1 + g;
  const R den = Elem<R>::fma((R)2 * g, u, a);
  const R rden = (R)1 / den;
  const R q = (a * b) * rden;
  const R omm = ((a * ((R)1 - u)) * rden) * (q + a);
  const R opm = ((b * u) * rden) * (q + b);
  mu = (R)0.5 * (opm - omm);
  s = std::sqrt(omm * opm);
}

// Rayleigh ("Rayleigh phase function for scattering of gases"):
// p(mu) = 3/8 (1 + mu^2); CDF(mu) = (mu^3 + 3 mu + 4)/8 = u.  Solve the cubic
// mu^3 + 3 mu - y = 0, y = 8u - 4, by 4 Newton steps from mu0 = y/4; sin(theta) = sqrt(1 - mu^2).
template <class R> inline void sample_rayleigh(R u, R& mu_out, R& s) {
  R y = Elem<R>::fma((R)8, u, (R)-4);
  R mu = (R)0.25 * y;
  for (int it = 0; it < 4; ++it) {
    R m2 = mu * mu;
    R fv = Elem<R>::fma(mu, m2, Elem<R>::fma((R)3, mu, -y));
    R dv = Elem<R>::fma((R)3, m2, (R)3);
    mu = mu - fv / dv;
  }
  mu = std::min((R)1, std::max((R)-1, mu));
  mu_out = mu;
  s = std::sqrt(std::max((R)0, Elem<R>::fma(-mu, mu, (R)1)));
}

// Rotate the unit direction (a,b,c) by the polar angle (cosine mu, sine s) and the azimuth (cphi,sphi); §3.9.
// r^2 = a^2 + b^2 is the squared sine of the direction's own polar angle (not 1 - c^2: no cancellation near the
// poles); below POLE_R2 the direction is taken as exactly +-z (an error below 1e-6 rad).  The result has norm
// 1 + O(rounding), so it is renormalised by the first-order reciprocal square root 3/2 - n2/2.
constexpr double POLE_R2 = 1e-12;
template <class R>
inline void rotate_dir(R& a, R& b, R& c, R mu, R s, R cphi, R sphi) {
  const R r2 = Elem<R>::fma(a, a, b * b);
  R nx, ny, nz;
  if (r2 > (R)POLE_R2) {
    const R r = std::sqrt(r2);
    const R ir = (R)1 / r;
    const R ah = a * ir, bh = b * ir;
    const R t1 = Elem<R>::fma(ah * c, cphi, -(bh * sphi));
    const R t2 = Elem<R>::fma(bh * c, cphi, ah * sphi);
    nx = Elem<R>::fma(s, t1, a * mu);
    ny = Elem<R>::fma(s, t2, b * mu);
    nz = Elem<R>::fma(-(s * r), cphi, c * mu);
  } else {
    nx = s * cphi; ny = s * sphi; nz = (c > 0 ? mu : -mu);
  }
  const R n2 = Elem<R>::fma(nz, nz, Elem<R>::fma(ny, ny, nx * nx));
  const R inv = Elem<R>::fma((R)-0.5, n2, (R)1.5);
  a = nx * inv; b = ny * inv; c = nz * inv;
}

}  // namespace

// ---------------------------------------------------------------------------
// C ABI (ctypes).  Counters mirror include/rt.h's rt_counters but are declared
// here independently.
// ---------------------------------------------------------------------------
extern "C" {

struct orc_counters {
  uint64_t n_photons, n_events, n_null, n_rayleigh, n_hg, n_atm_abs, n_sfc_hits, n_sfc_abs,
      n_toa, n_capped, n_cell_steps, n_relevel, n_roulette_killed, n_roulette_kept;
  int64_t capped_energy, roulette_lost, roulette_gained;
};

enum { ORC_ATM_ABS = 1, ORC_SFC_ABS = 2, ORC_TOD_EXIT = 3, ORC_CAPPED = 4, ORC_ROULETTE = 5 };

}  // extern "C"

namespace {

constexpr int64_t W0 = (int64_t)1 << 32;       // tally quanta per photon
constexpr uint32_t EVENT_CAP = 1u << 20;       // §3.12

struct Problem {
  int nx, ny, nz, bx, by, bz;
  int mx, my, mz;            // §3.5b: merged cells of mx x my x mz acceleration cells (1,1,1 = none)
  float merge_ratio;         // §3.5b: merged iff max c3 <= merge_ratio * min c3 over the merged cell's voxels
  int weighted;              // §3.14: 0 = analog absorption, 1 = the paper's weights + Russian roulette
  float diffuse_fraction;    // §3.15: share of photons launched diffusely (isotropic downwelling radiance)
  int sobol;                 // §3.15: entry points from a scrambled 2-D Sobol sequence instead of Philox
  float dx, dy, dz;
  const float *k_ext, *k_cloud, *ssa, *g, *albedo;
  double zenith_deg, azimuth_deg;
  uint64_t n_photons, first_id, seed;
  uint32_t stream_id;
  int64_t *atm_abs, *sfc_dir, *sfc_dif, *sfc_abs, *toa_up;
  int64_t* atm_abs_direct;   // optional (may be null): the part of atm_abs deposited by never-scattered photons
  uint32_t* records;
  double* margins;           // optional (may be null), one per photon: the smallest relative margin of any decision the
                             // photon took (bookkeeping only; no effect on the path).  A photon whose fp32 and fp64 paths
                             // differ must have met a decision whose two sides lie within rounding of each other.
  // optional decision log (may be null; bookkeeping only): the photon's first dlog_cap decisions, one byte each
  // (kind << 4 | outcome, kinds below) with the margin by which it was taken, and the number of decisions taken
  uint8_t* dlog_code; float* dlog_margin; uint32_t* dlog_count; uint32_t dlog_cap;
};

// decision kinds of the log: what was compared, and in which unit its margin is
enum { DK_COLLIDE = 1,   // tau <= k_hat t ?            distance between collision point and face, in face spacings of that axis
       DK_FACE = 2,      // which axis' face is next    distance to the runner-up face, in face spacings of the chosen axis
       DK_VOXEL = 3,     // floor to a voxel index      distance to the nearest voxel boundary, in voxels
       DK_CLASS = 4,     // absorb / HG / Rayleigh / null   distance to the nearest threshold, in units of k_hat
       DK_POLE = 5,      // which rotation formula      | |d_z| - threshold |
       DK_COLUMN = 6,    // floor to a surface column   as DK_VOXEL
       DK_ALBEDO = 7,    // u1 < albedo ?               |u1 - albedo|
       DK_RELEVEL = 8 }; // floor to a cell of the entered block (3.7b)   in cells

inline void add64(int64_t* p, int64_t v) { __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }

// §3.1 step 1: per-voxel cumulative coefficients, in Real, in this order.
template <class R> struct Vox { R c1, c2, c3, g; };
template <class R>
inline Vox<R> pack_voxel(float kf, float kcf, float wf, float gf) {
  R k = (R)kf, kc = (R)kcf, w = (R)wf;
  Vox<R> v;
  v.c3 = k;
  v.c1 = ((R)1 - w) * k;
  R frac = (k > 0) ? kc / k : (R)0;
  v.c2 = v.c1 + (w * k) * frac;
  v.c2 = std::min(v.c2, v.c3);
  v.c1 = std::min(v.c1, v.c2);
  v.g = (R)gf;
  return v;
}

// §3.15 point k of the 2-D Sobol sequence as 32-bit fractions: x1 = radical inverse of k in base 2,
// x2 = XOR of the direction numbers V0 = 2^31, Vj = Vj-1 ^ (Vj-1 >> 1) over the set bits j of k.
inline void sobol2(uint32_t k, uint32_t& x1, uint32_t& x2) {
  x1 = 0; x2 = 0;
  uint32_t V = 0x80000000u;
  for (int j = 0; j < 32; ++j) {
    if ((k >> j) & 1u) { x1 ^= 0x80000000u >> j; x2 ^= V; }
    V ^= V >> 1;
  }
}

template <class R>
void trace_range(const Problem& P, const std::vector<float>& khat, uint64_t i_begin, uint64_t i_end,
                 orc_counters& C) {
  typedef Elem<R> E;
  const int nx = P.nx, ny = P.ny, nz = P.nz, bx = P.bx, by = P.by, bz = P.bz;
  const int ncx = nx / bx, ncy = ny / by, ncz = nz / bz;
  const uint64_t ncol = (uint64_t)nx * ny;
  const uint64_t n_full = (P.n_photons / ncol) * ncol;
  const R dx = (R)P.dx, dy = (R)P.dy, dz = (R)P.dz;
  const R rdx = (R)1 / dx, rdy = (R)1 / dy, rdz = (R)1 / dz;
  // §3.5b/§3.7: cell extents at level 0 (one acceleration cell) and level 1 (a merged cell)
  const int mxyz[3] = {P.mx, P.my, P.mz};
  const R Lv[2][3] = {{(R)bx * dx, (R)by * dy, (R)bz * dz},
                      {(R)(P.mx * bx) * dx, (R)(P.my * by) * dy, (R)(P.mz * bz) * dz}};
  const R rL0[3] = {(R)1 / Lv[0][0], (R)1 / Lv[0][1], (R)1 / Lv[0][2]};   // §3.7b: reciprocal level-0 cell extents
  const int ncs[3] = {ncx, ncy, ncz};
  const R TINY = (R)1e-30f;

  // §3.3 sun direction: computed in double, then converted to Real.
  const double deg = 3.14159265358979323846 / 180.0;
  const double th = P.zenith_deg * deg, ph = P.azimuth_deg * deg;
  const R sun_x = (R)(float)(-std::sin(th) * std::sin(ph));
  const R sun_y = (R)(float)(-std::sin(th) * std::cos(ph));
  const R sun_z = (R)(float)(-std::cos(th));
  const uint32_t k0 = (uint32_t)P.seed, k1 = (uint32_t)(P.seed >> 32);

  for (uint64_t i = i_begin; i < i_end; ++i) {
    const uint64_t pid = P.first_id + i;
    const uint32_t p_lo = (uint32_t)pid, p_hi = (uint32_t)(pid >> 32);

    // ---- step 3: launch, event index 0 --------------------------------------
    U4 X = philox4x32_10(p_lo, p_hi, 0u, P.stream_id, k0, k1);
    R u0 = uni24<R>(X.x), u1 = uni24<R>(X.y), u2 = uni24<R>(X.z), u3 = uni24<R>(X.w);
    int ix, iy;
    if (i < n_full) {
      uint64_t col = i % ncol;
      ix = (int)(col % nx); iy = (int)(col / nx);
    } else {
      ix = std::min((int)(u2 * (R)nx), nx - 1);
      iy = std::min((int)(u3 * (R)ny), ny - 1);
    }
    if (P.sobol && i < n_full) {
      // §3.15 ("initialized at the domain top following a scrambled Sobol sequence"): within its column
      // the photon of pass k enters at point k of the 2-D Sobol sequence (radical inverse in base 2; second
      // coordinate from the direction numbers V0 = 2^31, Vj = Vj-1 ^ (Vj-1 >> 1)), scrambled by a random
      // digital shift (XOR) drawn per column, stream and call from Philox under the key (k0, k1 ^ 'SOBL')
      const uint32_t k = (uint32_t)(i / ncol), col32 = (uint32_t)(i % ncol);
      const U4 S = philox4x32_10(col32, P.stream_id, (uint32_t)P.first_id, (uint32_t)(P.first_id >> 32),
                                 k0, k1 ^ 0x534F424Cu);
      uint32_t x1, x2;
      sobol2(k, x1, x2);
      u0 = uni24<R>(x1 ^ S.x); u1 = uni24<R>(x2 ^ S.y);
    }
    int c[3] = {ix / bx, iy / by, ncz - 1};    // acceleration-cell index (at level 1: the merged cell's origin)
    // §3.5b: the sign bit of the stored majorant says whether the cell belongs to a merged cell
    auto load = [&](R& kh_out) {
      float s = khat[((size_t)c[2] * ncy + c[1]) * ncx + c[0]];
      kh_out = (R)std::fabs(s);
      return std::signbit(s) ? 1 : 0;
    };
    R kh;
    int lev = load(kh);
    if (lev) { c[0] -= c[0] % P.mx; c[1] -= c[1] % P.my; c[2] -= c[2] % P.mz; }
    // Position inside the current cell is carried as the REMAINING DISTANCES r[0..2] along the flight
    // direction to the cell's next face on each axis: a cell crossing subtracts the
    // smallest one from the other two and resets its own to the face spacing del = L |1/v| exactly, so
    // magnitudes never grow and rounding does not accumulate along a path.  Local coordinates are
    // recovered when needed as q = face - v r.
    R d[3] = {sun_x, sun_y, sun_z};            // unit direction
    bool direct = true;
    if (P.diffuse_fraction > 0.0f) {
      // §3.15 ("either along the sun beam or randomly generated, assuming isotropic downwelling diffuse
      // radiation at the TOD"): words of the Philox block at counter (id, 0 | 2^31): 0 decides, 1 and 2 give a
      // cosine-weighted downward direction (isotropic radiance: pdf(mu) = 2 mu)
      const U4 D = philox4x32_10(p_lo, p_hi, 0x80000000u, P.stream_id, k0, k1);
      if (uni24<R>(D.x) < (R)P.diffuse_fraction) {
        const R v1 = uni24<R>(D.y);
        const R mu = std::sqrt((R)1 - v1), sn = std::sqrt(v1);
        R sp, cp; E::sincos_2pi(uni24<R>(D.z), sp, cp);
        d[0] = sn * cp; d[1] = sn * sp; d[2] = -mu;
        direct = false;
      }
    }
    R v[3], iv[3];                             // nudged components and reciprocals
    R del[2][3];                               // distance between successive faces, per level and axis
    R r[3];                                    // remaining distance to the next face on each axis
    auto set_dir = [&]() {
      for (int a = 0; a < 3; ++a) {
        v[a] = (std::fabs(d[a]) < TINY) ? TINY : d[a];
        d[a] = v[a];                             // Q20 (round 2): the nudged component IS the direction from here on
        iv[a] = (R)1 / v[a];
        del[0][a] = Lv[0][a] * std::fabs(iv[a]);
        del[1][a] = Lv[1][a] * std::fabs(iv[a]);
      }
    };
    auto face = [&](int a) { return (v[a] > 0) ? Lv[lev][a] : (R)0; };
    auto place = [&](const R q[3]) {           // remaining distances from local coordinates
      for (int a = 0; a < 3; ++a) r[a] = (face(a) - q[a]) * iv[a];
    };
    auto local = [&](int a) {                  // local coordinate from a remaining distance
      return std::min(Lv[lev][a], std::max((R)0, E::fma(-v[a], r[a], face(a))));
    };
    set_dir();
    {
      const R q[3] = {((R)(ix % ((lev ? P.mx : 1) * bx)) + u0) * dx,
                      ((R)(iy % ((lev ? P.my : 1) * by)) + u1) * dy, Lv[lev][2]};
      place(q);
    }
    uint32_t e = 1, n_ev = 0, n_sc = 0, n_sfc = 0;
    int fate = 0; uint32_t term = 0;
    // decision margins (only when P.margins is given): how far each comparison or floor was from going the other way
    double mg = INFINITY;
    const bool track = P.margins != nullptr || P.dlog_code != nullptr;
    uint32_t n_dec = 0;
    auto note = [&](int kind, int outcome, double m) {
      if (m < mg) mg = m;
      if (P.dlog_code && n_dec < P.dlog_cap) {
        P.dlog_code[(size_t)i * P.dlog_cap + n_dec] = (uint8_t)((kind << 4) | (outcome & 15));
        P.dlog_margin[(size_t)i * P.dlog_cap + n_dec] = (float)m;
      }
      ++n_dec;
    };
    auto note_rel = [&](int kind, int outcome, R a, R b) {   // |a - b| relative to the larger magnitude
      const double s = std::max(std::fabs((double)a), std::fabs((double)b));
      note(kind, outcome, s > 0 ? std::fabs((double)a - (double)b) / s : 0.0);
    };
    auto note_floor = [&](int kind, int outcome, R f, int n) {   // f is floored to an index in 0..n-1: distance to the nearest interior boundary
      if (n <= 1) return;
      const double x = (double)f, k = std::min((double)(n - 1), std::max(1.0, std::round(x)));
      note(kind, outcome, std::fabs(x - k));
    };
    // §3.14 weighted mode: integer weight in tally quanta, W0 at launch.  Roulette (Iwabuchi 2006
    // as quoted in P:56): below W0/2 the photon survives with probability w/W0 exactly (a 32-bit word of
    // the Philox block at counter e | 2^31 is compared with w) and continues with W0, else it ends; both
    // branches go to a ledger so that energy closes exactly.  Returns true if the photon ended.
    uint64_t w = (uint64_t)W0;
    auto roulette = [&](uint32_t where) {
      if (w >= (uint64_t)W0 / 2) return false;
      const U4 Y = philox4x32_10(p_lo, p_hi, e | 0x80000000u, P.stream_id, k0, k1);
      if ((uint64_t)Y.w < w) { C.roulette_gained += W0 - (int64_t)w; ++C.n_roulette_kept; w = (uint64_t)W0; return false; }
      C.roulette_lost += (int64_t)w; ++C.n_roulette_killed; fate = ORC_ROULETTE; term = where;
      return true;
    };

    // ---- step 4: draw for event e -------------------------------------------
    R tau;
    auto draw = [&]() {
      X = philox4x32_10(p_lo, p_hi, e, P.stream_id, k0, k1);
      u0 = uni24<R>(X.x); u1 = uni24<R>(X.y); u2 = uni24<R>(X.z); u3 = uni24<R>(X.w);
      tau = E::neg_log_1m(u0);
    };
    draw();
    R rk = (kh > 0) ? (R)1 / kh : (R)0;
    const int bs[3] = {bx, by, bz};
    const R rds[3] = {rdx, rdy, rdz};

    while (fate == 0) {
      // ---- step 5: nearest face of the current cell; ties x < y < z -----------
      int axis; R t;
      if (r[0] <= r[1] && r[0] <= r[2]) { axis = 0; t = r[0]; }
      else if (r[1] <= r[2])            { axis = 1; t = r[1]; }
      else                              { axis = 2; t = r[2]; }
      R dtau = kh * t;
      if (track && kh > 0)                     // distance along the flight between the collision point and the face
        note(DK_COLLIDE, tau <= dtau ? 1 : 0, std::fabs((double)tau / (double)kh - (double)t) / (double)del[lev][axis]);
      if (kh > 0 && tau <= dtau) {
        // ---- step 7: tentative collision inside this cell -------------------
        R s = tau * rk;
        for (int a = 0; a < 3; ++a) r[a] = std::max((R)0, r[a] - s);
        R q[3]; int gv[3];
        for (int a = 0; a < 3; ++a) {
          q[a] = local(a);
          gv[a] = c[a] * bs[a] + std::min((int)(q[a] * rds[a]), (lev ? mxyz[a] : 1) * bs[a] - 1);
          if (track) note_floor(DK_VOXEL, gv[a], q[a] * rds[a], (lev ? mxyz[a] : 1) * bs[a]);
        }
        size_t vox = ((size_t)gv[2] * ny + gv[1]) * nx + gv[0];
        Vox<R> vx = pack_voxel<R>(P.k_ext[vox], P.k_cloud[vox], P.ssa[vox], P.g[vox]);
        ++n_ev; ++C.n_events;                  // step 6
        // ---- step 8: classify ----------------------------------------------
        R xi = u1 * kh;
        if (track) {
          const R x = P.weighted ? E::fma(u1, kh - vx.c1, vx.c1) : xi;
          const int cls = (!P.weighted && x < vx.c1) ? 0 : (x < vx.c2 ? 1 : (x < vx.c3 ? 2 : 3));
          double m = std::min(std::fabs((double)x - (double)vx.c2), std::fabs((double)x - (double)vx.c3));
          if (!P.weighted) m = std::min(m, std::fabs((double)x - (double)vx.c1));
          note(DK_CLASS, cls, m / (double)kh);
          if (cls == 1 || cls == 2) {            // which rotation formula (§3.9)
            const double r2 = (double)E::fma(d[0], d[0], d[1] * d[1]);
            note(DK_POLE, r2 > POLE_R2 ? 0 : 1, std::fabs(r2 - POLE_R2) / std::max(r2, POLE_R2));
          }
        }
        if (P.weighted) {
          // §3.14: deposit w * P(absorbed), P = c1 / k_hat as a 24-bit fixed-point number; the rest goes on
          const R f = vx.c1 * rk;
          const uint64_t pq = std::min<uint64_t>((uint64_t)1 << 24, (uint64_t)(f * (R)16777216.0));
          const uint64_t a = (w * pq) >> 24;
          if (a) add64(&P.atm_abs[vox], (int64_t)a);
          if (a && direct && P.atm_abs_direct) add64(&P.atm_abs_direct[vox], (int64_t)a);
          w -= a;
          if (w == 0) { ++C.n_atm_abs; fate = ORC_ATM_ABS; term = (uint32_t)vox; break; }
          xi = E::fma(u1, kh - vx.c1, vx.c1);     // what happens instead: uniform on [c1, k_hat)
        }
        if (!P.weighted && xi < vx.c1) {
          add64(&P.atm_abs[vox], W0); ++C.n_atm_abs;
          if (direct && P.atm_abs_direct) add64(&P.atm_abs_direct[vox], W0);
          fate = ORC_ATM_ABS; term = (uint32_t)vox; break;
        } else if (xi < vx.c2) {               // cloud droplet: Henyey-Greenstein
          R mu, sn; sample_hg<R>(vx.g, u2, mu, sn);
          R sp, cp; E::sincos_2pi(u3, sp, cp);
          rotate_dir<R>(d[0], d[1], d[2], mu, sn, cp, sp); set_dir(); place(q);
          direct = false; ++n_sc; ++C.n_hg;
        } else if (xi < vx.c3) {               // gas: Rayleigh
          R mu, sn; sample_rayleigh<R>(u2, mu, sn);
          R sp, cp; E::sincos_2pi(u3, sp, cp);
          rotate_dir<R>(d[0], d[1], d[2], mu, sn, cp, sp); set_dir(); place(q);
          direct = false; ++n_sc; ++C.n_rayleigh;
        } else {
          ++C.n_null;                          // null collision: direction unchanged
        }
        if (P.weighted && roulette((uint32_t)vox)) break;
        ++e;
        if (e > EVENT_CAP) {                   // step 12
          ++C.n_capped; C.capped_energy += P.weighted ? (int64_t)w : W0; fate = ORC_CAPPED; term = 0; break;
        }
        draw();
      } else {
        // ---- step 5 (cont.): leave the cell through `axis` -------------------
        if (track) {                           // which face: the gap to the runner-up
          const R o1 = r[(axis + 1) % 3], o2 = r[(axis + 2) % 3];
          note(DK_FACE, axis, std::fabs((double)std::min(o1, o2) - (double)t) / (double)del[lev][axis]);
        }
        tau = tau - dtau;
        ++C.n_cell_steps;
        const int step = lev ? mxyz[axis] : 1;
        for (int a = 0; a < 3; ++a) r[a] = (a == axis) ? del[lev][a] : r[a] - t;
        bool at_sfc = false, at_top = false;
        if (v[axis] > 0) {
          c[axis] += step;
          if (c[axis] >= ncs[axis]) { if (axis == 2) at_top = true; else c[axis] -= ncs[axis]; }
        } else {
          c[axis] -= step;
          if (c[axis] < 0) { if (axis == 2) at_sfc = true; else c[axis] += ncs[axis]; }
        }
        if (at_sfc || at_top) {
          R qx = local(0), qy = local(1);
          int hx = c[0] * bx + std::min((int)(qx * rdx), (lev ? P.mx : 1) * bx - 1);
          int hy = c[1] * by + std::min((int)(qy * rdy), (lev ? P.my : 1) * by - 1);
          if (track) { note_floor(DK_COLUMN, hx, qx * rdx, (lev ? P.mx : 1) * bx); note_floor(DK_COLUMN, hy, qy * rdy, (lev ? P.my : 1) * by); }
          size_t col = (size_t)hy * nx + hx;
          if (at_top) {                        // step 11
            add64(&P.toa_up[col], P.weighted ? (int64_t)w : W0); ++C.n_toa;
            fate = ORC_TOD_EXIT; term = (uint32_t)col; break;
          }
          // ---- step 10: Lambertian surface ---------------------------------
          ++C.n_sfc_hits; ++n_sfc;
          add64(direct ? &P.sfc_dir[col] : &P.sfc_dif[col], P.weighted ? (int64_t)w : W0);
          bool reflect;
          if (P.weighted) {
            // §3.14: the albedo reduces the weight, 24-bit fixed point; always reflect
            const uint64_t aq = std::min<uint64_t>((uint64_t)1 << 24, (uint64_t)((R)P.albedo[col] * (R)16777216.0));
            const uint64_t refl = (w * aq) >> 24;
            if (w - refl) add64(&P.sfc_abs[col], (int64_t)(w - refl));
            w = refl;
            if (w == 0) { ++C.n_sfc_abs; fate = ORC_SFC_ABS; term = (uint32_t)col; break; }
            if (roulette((uint32_t)col)) break;
            reflect = true;
          } else {
            reflect = u1 < (R)P.albedo[col];
            if (track) note(DK_ALBEDO, reflect ? 1 : 0, std::fabs((double)u1 - (double)P.albedo[col]));
          }
          if (reflect) {
            R mu = std::sqrt((R)1 - u2), s = std::sqrt(u2);
            R sp, cp; E::sincos_2pi(u3, sp, cp);
            d[0] = s * cp; d[1] = s * sp; d[2] = mu; set_dir();
            direct = false; c[2] = 0;          // back in the cell it left (level unchanged)
            const R q[3] = {qx, qy, (R)0};
            place(q);
            ++e;
            if (e > EVENT_CAP) {
              ++C.n_capped; C.capped_energy += P.weighted ? (int64_t)w : W0; fate = ORC_CAPPED; term = 0; break;
            }
            draw();
          } else {
            add64(&P.sfc_abs[col], W0); ++C.n_sfc_abs;
            fate = ORC_SFC_ABS; term = (uint32_t)col; break;
          }
        } else {
          // ---- §3.7b: the entered cell's level; change of level at a merged cell's face ------
          const int lev_new = load(kh);
          if (lev_new != lev) {
            ++C.n_relevel;
            if (lev_new == 1) {
              // into a merged cell: distances to ITS faces; the index becomes its origin
              for (int a = 0; a < 3; ++a) {
                const int m = mxyz[a], o = c[a] % m;
                if (a != axis) {
                  const int n = (v[a] > 0) ? (m - 1 - o) : o;   // whole cells between here and that face
                  r[a] = E::fma((R)n, del[0][a], r[a]);
                } else {
                  r[a] = del[1][a];
                }
                c[a] -= o;
              }
            } else {
              // out of a merged cell into single cells: which cell of the entered block, and the
              // distance to that cell's faces
              for (int a = 0; a < 3; ++a) {
                const int m = mxyz[a];
                if (a != axis) {
                  // whole level-0 cells in r: r / del^0 with del^0 = L^0 |1/v|, taken as r (|v| (1/L^0))
                  const R cells = r[a] * (std::fabs(v[a]) * rL0[a]);
                  const int k = std::min(m - 1, (int)cells);
                  if (track) note_floor(DK_RELEVEL, k, cells, m);
                  r[a] = std::max((R)0, E::fma(-(R)k, del[0][a], r[a]));
                  c[a] += (v[a] > 0) ? (m - 1 - k) : k;
                } else {
                  r[a] = del[0][a];
                  if (!(v[a] > 0)) c[a] += m - 1;               // entered through the block's far side
                }
              }
              load(kh);                                          // the single cell's own majorant
            }
            lev = lev_new;
          }
        }
        rk = (kh > 0) ? (R)1 / kh : (R)0;
      }
    }
    ++C.n_photons;
    if (P.margins) P.margins[i] = mg;
    if (P.dlog_count) P.dlog_count[i] = n_dec;
    if (P.records) {
      uint32_t* r = P.records + 4 * i;
      r[0] = (uint32_t)fate | (std::min(n_sfc, 0xFFFFFFu) << 8);
      r[1] = term; r[2] = n_ev; r[3] = n_sc;
    }
  }
}

// §3.5 majorant: highest extinction coefficient within each acceleration cell.
// §3.5b merged cells: blocks of mx x my x mz acceleration cells whose voxels all have nearly the same
// extinction (max <= merge_ratio * min, one fp32 multiply) are traversed as ONE cell with the block's
// maximum; every cell of such a block stores -(block maximum) (sign bit set, also for 0).
std::vector<float> build_majorant(const Problem& P) {
  const int ncx = P.nx / P.bx, ncy = P.ny / P.by, ncz = P.nz / P.bz;
  std::vector<float> kh((size_t)ncx * ncy * ncz, 0.0f);
  for (int z = 0; z < P.nz; ++z)
    for (int y = 0; y < P.ny; ++y)
      for (int x = 0; x < P.nx; ++x) {
        float k = P.k_ext[((size_t)z * P.ny + y) * P.nx + x];
        float& m = kh[((size_t)(z / P.bz) * ncy + (y / P.by)) * ncx + (x / P.bx)];
        if (k > m) m = k;
      }
  if (P.mx * P.my * P.mz == 1) return kh;
  const int sx = P.mx * P.bx, sy = P.my * P.by, sz = P.mz * P.bz;   // merged-cell extent in voxels
  for (int Z = 0; Z < P.nz / sz; ++Z)
    for (int Y = 0; Y < P.ny / sy; ++Y)
      for (int X = 0; X < P.nx / sx; ++X) {
        float kmax = 0.0f, kmin = INFINITY;
        for (int z = Z * sz; z < (Z + 1) * sz; ++z)
          for (int y = Y * sy; y < (Y + 1) * sy; ++y)
            for (int x = X * sx; x < (X + 1) * sx; ++x) {
              float k = P.k_ext[((size_t)z * P.ny + y) * P.nx + x];
              kmax = std::max(kmax, k); kmin = std::min(kmin, k);
            }
        if (!(kmax <= P.merge_ratio * kmin)) continue;
        for (int cz = Z * P.mz; cz < (Z + 1) * P.mz; ++cz)
          for (int cy = Y * P.my; cy < (Y + 1) * P.my; ++cy)
            for (int cx = X * P.mx; cx < (X + 1) * P.mx; ++cx)
              kh[((size_t)cz * ncy + cy) * ncx + cx] = -kmax;
      }
  return kh;
}

}  // namespace

extern "C" {

// Returns 0 on success, -1 on bad arguments.  Tallies and counters are ADDED to.
// elapsed_s (may be NULL) receives the wall time of the photon loop only.
int orc_trace(int precision, int nx, int ny, int nz, float dx, float dy, float dz, int bx, int by,
              int bz, int mx, int my, int mz, float merge_ratio, int weighted, float diffuse_fraction,
              int sobol, const float* k_ext, const float* k_ext_cloud, const float* ssa, const float* g,
              const float* sfc_albedo, double zenith_deg, double azimuth_deg, uint64_t n_photons,
              uint64_t first_photon_id, uint64_t seed, uint32_t stream_id, int64_t* atm_abs,
              int64_t* sfc_dir, int64_t* sfc_dif, int64_t* sfc_abs, int64_t* toa_up,
              int64_t* atm_abs_direct, orc_counters* counters, uint32_t* records, int n_threads, double* elapsed_s,
              double* margins, uint64_t range_begin, uint64_t range_count,
              uint8_t* dlog_code, float* dlog_margin, uint32_t* dlog_count, uint32_t dlog_cap) {
  if (nx <= 0 || ny <= 0 || nz <= 0 || bx <= 0 || by <= 0 || bz <= 0) return -1;
  if (nx % bx || ny % by || nz % bz) return -1;
  if (mx <= 0 || my <= 0 || mz <= 0 || (nx / bx) % mx || (ny / by) % my || (nz / bz) % mz) return -1;
  if (!(zenith_deg >= 0.0 && zenith_deg < 90.0)) return -1;
  if (precision != 32 && precision != 64) return -1;
  if (!(diffuse_fraction >= 0.0f && diffuse_fraction <= 1.0f)) return -1;
  Problem P{nx, ny, nz, bx, by, bz, mx, my, mz, merge_ratio, weighted ? 1 : 0, diffuse_fraction, sobol ? 1 : 0, dx, dy, dz, k_ext, k_ext_cloud, ssa, g, sfc_albedo,
            zenith_deg, azimuth_deg, n_photons, first_photon_id, seed, stream_id,
            atm_abs, sfc_dir, sfc_dif, sfc_abs, toa_up, atm_abs_direct, records, margins,
            dlog_code, dlog_margin, dlog_count, dlog_cap};
  // a PART of the job: photon indices [range_begin, range_begin + range_count) of the n_photons;
  // records and margins stay indexed by the index in the job
  if (range_begin > n_photons || range_count > n_photons - range_begin) return -1;
  std::vector<float> khat = build_majorant(P);
  if (n_threads < 1) n_threads = 1;
  std::vector<orc_counters> cs(n_threads);
  std::memset(cs.data(), 0, sizeof(orc_counters) * n_threads);
  auto run = [&](int t) {
    uint64_t b = range_begin + range_count * (uint64_t)t / n_threads, e = range_begin + range_count * (uint64_t)(t + 1) / n_threads;
    if (precision == 64) trace_range<double>(P, khat, b, e, cs[t]);
    else                 trace_range<float>(P, khat, b, e, cs[t]);
  };
  auto t0 = std::chrono::steady_clock::now();
  if (n_threads == 1) run(0);
  else {
    std::vector<std::thread> th;
    for (int t = 0; t < n_threads; ++t) th.emplace_back(run, t);
    for (auto& x : th) x.join();
  }
  auto t1 = std::chrono::steady_clock::now();
  if (elapsed_s) *elapsed_s = std::chrono::duration<double>(t1 - t0).count();
  if (counters) {
    uint64_t* dst = (uint64_t*)counters;
    for (int t = 0; t < n_threads; ++t) {
      const uint64_t* src = (const uint64_t*)&cs[t];
      for (size_t j = 0; j < sizeof(orc_counters) / 8; ++j) dst[j] += src[j];
    }
  }
  return 0;
}

// ---- small exports so the pins in tests/ can reach each part by itself ----
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  U4 r = philox4x32_10(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1]);
  out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
void orc_neg_log_f32(const float* w, float* out, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) out[i] = spec_neg_log(w[i]);
}
void orc_sincos_2pi_f32(const float* u, float* sn, float* cs, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) spec_sincos_2pi(u[i], sn[i], cs[i]);
}
// mu and sin(theta) for each u (sn may be NULL)
void orc_sample_hg(int precision, double g, const double* u, double* mu, double* sn, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) {
    if (precision == 64) { double m, s; sample_hg<double>(g, u[i], m, s); mu[i] = m; if (sn) sn[i] = s; }
    else { float m, s; sample_hg<float>((float)g, (float)u[i], m, s); mu[i] = m; if (sn) sn[i] = s; }
  }
}
void orc_sample_rayleigh(int precision, const double* u, double* mu, double* sn, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) {
    if (precision == 64) { double m, s; sample_rayleigh<double>(u[i], m, s); mu[i] = m; if (sn) sn[i] = s; }
    else { float m, s; sample_rayleigh<float>((float)u[i], m, s); mu[i] = m; if (sn) sn[i] = s; }
  }
}
// d is 3 doubles in/out; rotation by the polar angle (cosine mu, sine sn) and azimuth 2*pi*u_phi.
void orc_rotate(int precision, double* d, double mu, double sn, double u_phi) {
  if (precision == 64) {
    double s, c; Elem<double>::sincos_2pi(u_phi, s, c);
    rotate_dir<double>(d[0], d[1], d[2], mu, sn, c, s);
  } else {
    float a = (float)d[0], b = (float)d[1], cc = (float)d[2], s, c;
    Elem<float>::sincos_2pi((float)u_phi, s, c);
    rotate_dir<float>(a, b, cc, (float)mu, (float)sn, c, s);
    d[0] = a; d[1] = b; d[2] = cc;
  }
}
// c is 4 floats out per voxel: c1, c2, c3, g (fp32 packing, step 1).
void orc_pack_optics_f32(const float* k, const float* kc, const float* w, const float* g, float* c,
                         uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) {
    Vox<float> v = pack_voxel<float>(k[i], kc[i], w[i], g[i]);
    c[4 * i] = v.c1; c[4 * i + 1] = v.c2; c[4 * i + 2] = v.c3; c[4 * i + 3] = v.g;
  }
}
void orc_majorant(int nx, int ny, int nz, int bx, int by, int bz, int mx, int my, int mz,
                  float merge_ratio, const float* k_ext, float* out) {
  Problem P{}; P.nx = nx; P.ny = ny; P.nz = nz; P.bx = bx; P.by = by; P.bz = bz; P.k_ext = k_ext;
  P.mx = mx; P.my = my; P.mz = mz; P.merge_ratio = merge_ratio;
  std::vector<float> kh = build_majorant(P);
  std::memcpy(out, kh.data(), kh.size() * sizeof(float));
}
void orc_sobol2(const uint32_t* k, uint32_t* x1, uint32_t* x2, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) sobol2(k[i], x1[i], x2[i]);
}
int orc_hardware_threads() { return (int)std::thread::hardware_concurrency(); }

}  // extern "C"
