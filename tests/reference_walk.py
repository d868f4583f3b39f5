"""An INDEPENDENT brute-force photon walker for tests (pure Python, fp64): DESIGN.md §3 restated the plain way.

Why it exists: the oracle's fp32 instantiation follows the same normative text as the CUDA
kernel, remaining-distance traversal and two-level merged cells included, so a mistake in that text's traversal or
level-change arithmetic would be made on both sides.  This walker shares none of it:
  * positions are plain GLOBAL coordinates in metres (unwrapped: the cell index runs over all integers and is
    wrapped only to look the majorant up), not remaining distances;
  * it knows no levels: it walks level-0 acceleration cells one by one everywhere and only reads, per cell, the
    majorant VALUE that DESIGN.md §3.5/§3.5b define (cell maximum, or the block maximum inside a merged block), built
    here with numpy reshapes.  Null-collision tracking through a piecewise-constant majorant gives the same collision
    points however the constant pieces are cut, so its photons must equal the oracle's, event by event;
  * its own Philox4x32-10, its own samplers and rotation typed from §3.9 (no fma: differences of 1e-16).
Against the fp64 oracle the per-photon records (fate, terminal bin, events, scatters, surface hits) must be equal for
every photon up to decisions that tie within ~1e-12, i.e. for all of a few thousand photons.  Slow by design
(~1 ms per photon); analog mode, Philox entry points, direct beam only.
"""
import math

import numpy as np

M0, M1, W0K, W1K = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
MASK = 0xFFFFFFFF
W0 = 1 << 32
TINY = float(np.float32(1e-30))
EVENT_CAP = 1 << 20


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    for _ in range(10):
        p0 = M0 * c0
        p1 = M1 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & MASK, p1 & MASK, ((p0 >> 32) ^ c3 ^ k1) & MASK, p0 & MASK
        k0 = (k0 + W0K) & MASK
        k1 = (k1 + W1K) & MASK
    return c0, c1, c2, c3


def u24(x):
    return (x >> 8) / 16777216.0


def majorant_values(k_ext, block, merge=(1, 1, 1), ratio=1.25):
    """Per level-0 cell: the majorant DESIGN.md §3.5 / §3.5b give it (float64 array [ncz][ncy][ncx])."""
    nz, ny, nx = k_ext.shape
    bx, by, bz = block
    k = k_ext.astype(np.float32)
    cells = k.reshape(nz // bz, bz, ny // by, by, nx // bx, bx)
    kh = cells.max(axis=(1, 3, 5)).astype(np.float64)
    mx, my, mz = merge
    if mx * my * mz > 1:
        sz, sy, sx = mz * bz, my * by, mx * bx
        blocks = k.reshape(nz // sz, sz, ny // sy, sy, nx // sx, sx)
        hi = blocks.max(axis=(1, 3, 5))
        lo = blocks.min(axis=(1, 3, 5))
        merged = hi <= np.float32(ratio) * lo                    # one fp32 multiply, as §3.5b says
        hi_c = np.repeat(np.repeat(np.repeat(hi, mz, 0), my, 1), mx, 2).astype(np.float64)
        mg_c = np.repeat(np.repeat(np.repeat(merged, mz, 0), my, 1), mx, 2)
        kh = np.where(mg_c, hi_c, kh)
    return kh


def walk(grid, optics, zenith_deg, azimuth_deg, n_photons, seed=1, stream_id=0, first_photon_id=0,
         merge=(1, 1, 1), merge_ratio=1.25):
    """Trace n_photons photons; returns (records uint32 [n][4], tallies dict of int64 arrays, counters dict)."""
    nx, ny, nz, dx, dy, dz, bx, by, bz = grid
    dx, dy, dz = float(np.float32(dx)), float(np.float32(dy)), float(np.float32(dz))
    kx = np.ascontiguousarray(optics["k_ext"], dtype=np.float32).reshape(nz, ny, nx)
    kc = np.ascontiguousarray(optics["k_ext_cloud"], dtype=np.float32).reshape(nz, ny, nx)
    ww = np.ascontiguousarray(optics["ssa"], dtype=np.float32).reshape(nz, ny, nx)
    gg = np.ascontiguousarray(optics["g"], dtype=np.float32).reshape(nz, ny, nx)
    alb = np.ascontiguousarray(optics["sfc_albedo"], dtype=np.float32).reshape(ny, nx)
    khat = majorant_values(kx, (bx, by, bz), merge, merge_ratio)
    ncx, ncy, ncz = nx // bx, ny // by, nz // bz
    Lc = (bx * dx, by * dy, bz * dz)                             # level-0 cell extent
    ncol = nx * ny
    n_full = (n_photons // ncol) * ncol
    th, ph = math.radians(zenith_deg), math.radians(azimuth_deg)
    sun = [float(np.float32(-math.sin(th) * math.sin(ph))), float(np.float32(-math.sin(th) * math.cos(ph))),
           float(np.float32(-math.cos(th)))]
    k0, k1 = seed & MASK, (seed >> 32) & MASK
    tal = {"atm_abs": np.zeros((nz, ny, nx), np.int64), "sfc_dir": np.zeros((ny, nx), np.int64),
           "sfc_dif": np.zeros((ny, nx), np.int64), "sfc_abs": np.zeros((ny, nx), np.int64),
           "toa_up": np.zeros((ny, nx), np.int64)}
    cnt = dict(n_events=0, n_null=0, n_hg=0, n_rayleigh=0, n_atm_abs=0, n_sfc_hits=0, n_sfc_abs=0, n_toa=0, n_cell_steps=0)
    rec = np.zeros((n_photons, 4), np.uint32)

    def nudge(d):
        return [TINY if abs(c) < TINY else c for c in d]

    for i in range(n_photons):
        pid = first_photon_id + i
        plo, phi = pid & MASK, (pid >> 32) & MASK
        x0, x1, x2, x3 = philox4x32_10(plo, phi, 0, stream_id, k0, k1)
        if i < n_full:
            col = i % ncol
            ix, iy = col % nx, col // nx
        else:
            ix, iy = min(int(u24(x2) * nx), nx - 1), min(int(u24(x3) * ny), ny - 1)
        p = [(ix + u24(x0)) * dx, (iy + u24(x1)) * dy, nz * dz]  # global, unwrapped
        c = [ix // bx, iy // by, ncz - 1]                        # level-0 cell, unwrapped in x and y
        d = nudge(sun)
        direct, e, n_ev, n_sc, n_sfc, fate, term = True, 1, 0, 0, 0, 0, 0
        while fate == 0:
            w0, w1, w2, w3 = philox4x32_10(plo, phi, e, stream_id, k0, k1)
            tau = -math.log(1.0 - u24(w0))
            u1 = u24(w1)
            # ---- one flight: cell by cell until the optical depth is used up or the domain is left ----
            while True:
                kh = khat[c[2], c[1] % ncy, c[0] % ncx]
                best, t = 0, math.inf
                for a in range(3):
                    face = (c[a] + 1) * Lc[a] if d[a] > 0 else c[a] * Lc[a]
                    ta = (face - p[a]) / d[a]
                    if ta < t:                                   # strict: ties go to the lower axis
                        best, t = a, ta
                t = max(t, 0.0)
                if kh > 0 and tau <= kh * t:
                    s = tau / kh
                    p = [p[a] + d[a] * s for a in range(3)]
                    arrived = None
                    break
                tau -= kh * t
                cnt["n_cell_steps"] += 1
                p = [p[a] + d[a] * t for a in range(3)]
                if d[best] > 0:
                    c[best] += 1
                    p[best] = c[best] * Lc[best]                 # exactly on the face
                else:
                    p[best] = c[best] * Lc[best]
                    c[best] -= 1
                if best == 2 and (c[2] < 0 or c[2] >= ncz):
                    arrived = "sfc" if c[2] < 0 else "top"
                    break
            if arrived is None:
                # ---- tentative collision: the voxel of the point, inside the cell ----
                v = []
                for a, (dd, b, nn) in enumerate(((dx, bx, nx), (dy, by, ny), (dz, bz, nz))):
                    g = int(math.floor(p[a] / dd))
                    g = min(max(g, c[a] * b), c[a] * b + b - 1)
                    v.append(g % nn if a < 2 else g)
                vx, vy, vz = v
                k = float(kx[vz, vy, vx])
                w = float(ww[vz, vy, vx])
                c3 = k
                c1 = (1.0 - w) * k
                c2 = c1 + (w * k) * (float(kc[vz, vy, vx]) / k if k > 0 else 0.0)
                c2 = min(c2, c3)
                c1 = min(c1, c2)
                n_ev += 1
                cnt["n_events"] += 1
                xi = u1 * kh
                if xi < c1:
                    tal["atm_abs"][vz, vy, vx] += W0
                    cnt["n_atm_abs"] += 1
                    fate, term = 1, (vz * ny + vy) * nx + vx
                    break
                if xi < c3:
                    u2, u3 = u24(w2), u24(w3)
                    if xi < c2:                                  # cloud droplet: Henyey-Greenstein, §3.9
                        g_ = float(gg[vz, vy, vx])
                        a_, b_ = 1.0 - g_, 1.0 + g_
                        den = 2.0 * g_ * u2 + a_
                        q = a_ * b_ / den
                        omm = a_ * (1.0 - u2) / den * (q + a_)
                        opm = b_ * u2 / den * (q + b_)
                        mu, sn = 0.5 * (opm - omm), math.sqrt(omm * opm)
                        cnt["n_hg"] += 1
                    else:                                        # gas: Rayleigh, cubic solved in closed form
                        qq = 4.0 * u2 - 2.0
                        A = (qq + math.sqrt(qq * qq + 1.0)) ** (1.0 / 3.0)
                        mu = min(1.0, max(-1.0, A - 1.0 / A))
                        sn = math.sqrt(max(0.0, 1.0 - mu * mu))
                        cnt["n_rayleigh"] += 1
                    cp, sp = math.cos(2 * math.pi * u3), math.sin(2 * math.pi * u3)
                    a0, b0, c0 = d
                    r2 = a0 * a0 + b0 * b0
                    if r2 > 1e-12:
                        r = math.sqrt(r2)
                        ah, bh = a0 / r, b0 / r
                        nd = [sn * (ah * c0 * cp - bh * sp) + a0 * mu, sn * (bh * c0 * cp + ah * sp) + b0 * mu,
                              -sn * r * cp + c0 * mu]
                    else:
                        nd = [sn * cp, sn * sp, mu if c0 > 0 else -mu]
                    n2 = nd[0] * nd[0] + nd[1] * nd[1] + nd[2] * nd[2]
                    inv = 1.5 - 0.5 * n2
                    d = nudge([x * inv for x in nd])
                    direct = False
                    n_sc += 1
                else:
                    cnt["n_null"] += 1
            elif arrived == "top":
                hx, hy = int(math.floor(p[0] / dx)), int(math.floor(p[1] / dy))
                hx = min(max(hx, c[0] * bx), c[0] * bx + bx - 1) % nx
                hy = min(max(hy, c[1] * by), c[1] * by + by - 1) % ny
                tal["toa_up"][hy, hx] += W0
                cnt["n_toa"] += 1
                fate, term = 3, hy * nx + hx
                break
            else:
                hx, hy = int(math.floor(p[0] / dx)), int(math.floor(p[1] / dy))
                hx = min(max(hx, c[0] * bx), c[0] * bx + bx - 1) % nx
                hy = min(max(hy, c[1] * by), c[1] * by + by - 1) % ny
                n_sfc += 1
                cnt["n_sfc_hits"] += 1
                tal["sfc_dir" if direct else "sfc_dif"][hy, hx] += W0
                if u1 < float(alb[hy, hx]):
                    u2, u3 = u24(w2), u24(w3)
                    mu, sn = math.sqrt(1.0 - u2), math.sqrt(u2)
                    d = nudge([sn * math.cos(2 * math.pi * u3), sn * math.sin(2 * math.pi * u3), mu])
                    direct = False
                    c[2] = 0
                    p[2] = 0.0
                else:
                    tal["sfc_abs"][hy, hx] += W0
                    cnt["n_sfc_abs"] += 1
                    fate, term = 2, hy * nx + hx
                    break
            e += 1
            if e > EVENT_CAP:
                fate, term = 4, 0
        rec[i] = (fate | (min(n_sfc, 0xFFFFFF) << 8), term, n_ev, n_sc)
    return rec, tal, cnt
