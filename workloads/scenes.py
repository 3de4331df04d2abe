"""Synthetic scenes behind the workload generators: a sphere union (config 2) and a box room
with random boxes and spheres seen by pinhole keyframes (configs 3-5).  Input generation only
(analytic ray casting, shading, noise); no arithmetic of the method lives here."""
import numpy as np


def pack_bits(mask_flat):
    """bool[G^3] in canonical order i = gx + G*(gy + G*gz) -> uint8[G^3/8], bit i&7 of byte i>>3."""
    return np.packbits(np.asarray(mask_flat, dtype=np.uint8), bitorder="little")


def cell_centres_axis(G):
    return (np.arange(G, dtype=np.float64) + 0.5) / G


# ------------------------------------------------------------------------------ sphere union

def inside_any_sphere(p, centres, radii):
    inside = np.zeros(p.shape[0], bool)
    for c, r in zip(centres, radii):
        inside |= ((p - c) ** 2).sum(1) < r * r
    return inside


def sphere_union_occupancy(rng, G, target_fraction):
    """Append spheres (centre ~ U[0.1,0.9]^3, radius ~ U[0.04,0.12]) until >= target_fraction of
    the G^3 cell centres are covered; bit = centre inside any sphere."""
    ax = cell_centres_axis(G)
    zz, yy, xx = np.meshgrid(ax, ax, ax, indexing="ij")      # index [gz, gy, gx]
    mask = np.zeros((G, G, G), bool)
    centres, radii = [], []
    while mask.mean() < target_fraction:
        c = rng.uniform(0.1, 0.9, 3)
        r = rng.uniform(0.04, 0.12)
        centres.append(c)
        radii.append(r)
        lo = np.clip(np.floor((c - r) * G).astype(int), 0, G - 1)
        hi = np.clip(np.ceil((c + r) * G).astype(int) + 1, 1, G)
        sl = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
        d2 = (xx[sl] - c[0]) ** 2 + (yy[sl] - c[1]) ** 2 + (zz[sl] - c[2]) ** 2
        mask[sl] |= d2 < r * r
    return np.array(centres), np.array(radii), pack_bits(mask.reshape(-1)), float(mask.mean())


def ray_sphere_union(o, d, centres, radii):
    """First positive hit distance of unit-direction rays with the union (inf if none)."""
    best = np.full(o.shape[0], np.inf)
    for c, r in zip(centres, radii):
        oc = o - c
        b = (oc * d).sum(1)
        cc = (oc * oc).sum(1) - r * r
        disc = b * b - cc
        ok = disc >= 0
        sq = np.sqrt(np.where(ok, disc, 0.0))
        t0, t1 = -b - sq, -b + sq
        t = np.where(t0 > 1e-9, t0, np.where(t1 > 1e-9, t1, np.inf))
        best = np.where(ok & (t < best), t, best)
    return best


# ------------------------------------------------------------------------------------- room

class Room:
    """Box room [0,8]x[0,6]x[0,3] m seen from inside, plus 10 axis-aligned boxes (side ~
    U[0.3,1.5]) and 10 spheres (radius ~ U[0.2,0.7]); every surface has an albedo ~ U[0.2,0.9]^3;
    a point light sits at the room centre near the ceiling."""
    size = np.array([8.0, 6.0, 3.0])

    def __init__(self, seed):
        rng = np.random.Generator(np.random.PCG64([seed, 0x5c3e]))
        self.box_lo, self.box_hi = [], []
        for _ in range(10):
            side = rng.uniform(0.3, 1.5, 3)
            c = rng.uniform(0.0, 1.0, 3) * self.size
            self.box_lo.append(np.maximum(c - side / 2, 0.0))
            self.box_hi.append(np.minimum(c + side / 2, self.size))
        self.sph_c = [rng.uniform(0.0, 1.0, 3) * self.size for _ in range(10)]
        self.sph_r = [rng.uniform(0.2, 0.7) for _ in range(10)]
        self.albedo = rng.uniform(0.2, 0.9, (6 + 20, 3))
        self.light = np.array([4.0, 3.0, 2.8])

    def inside_primitive(self, p):
        inside = np.zeros(p.shape[0], bool)
        for lo, hi in zip(self.box_lo, self.box_hi):
            inside |= np.all((p > lo) & (p < hi), axis=1)
        for c, r in zip(self.sph_c, self.sph_r):
            inside |= ((p - c) ** 2).sum(1) < r * r
        return inside

    def cast(self, o, d):
        """Analytic ray cast.  Returns (range, normal[.,3], surface id)."""
        n = o.shape[0]
        best = np.full(n, np.inf)
        normal = np.zeros((n, 3))
        sid = np.zeros(n, np.int64)
        with np.errstate(divide="ignore", invalid="ignore"):
            inv = 1.0 / d
            # the six walls, from inside: the exit point of the room slab
            for ax in range(3):
                for side, plane in ((0, 0.0), (1, self.size[ax])):
                    t = (plane - o[:, ax]) * inv[:, ax]
                    p = o + t[:, None] * d
                    ok = (t > 1e-9) & np.all((p >= -1e-9) & (p <= self.size + 1e-9), axis=1)
                    ok &= (d[:, ax] < 0) if side == 0 else (d[:, ax] > 0)
                    upd = ok & (t < best)
                    best = np.where(upd, t, best)
                    nn = np.zeros(3)
                    nn[ax] = 1.0 if side == 0 else -1.0
                    normal[upd] = nn
                    sid[upd] = 2 * ax + side
            # boxes: slab test
            for i, (lo, hi) in enumerate(zip(self.box_lo, self.box_hi)):
                t0 = (lo - o) * inv
                t1 = (hi - o) * inv
                tn = np.minimum(t0, t1)
                tf = np.maximum(t0, t1)
                tnear = np.nanmax(tn, axis=1)
                tfar = np.nanmin(tf, axis=1)
                ok = (tnear <= tfar) & (tnear > 1e-9)
                upd = ok & (tnear < best)
                if upd.any():
                    ax = np.nanargmax(tn, axis=1)
                    nn = np.zeros((n, 3))
                    nn[np.arange(n), ax] = -np.sign(d[np.arange(n), ax])
                    best = np.where(upd, tnear, best)
                    normal[upd] = nn[upd]
                    sid[upd] = 6 + i
            # spheres: quadratic
            for i, (c, r) in enumerate(zip(self.sph_c, self.sph_r)):
                oc = o - c
                b = (oc * d).sum(1)
                disc = b * b - ((oc * oc).sum(1) - r * r)
                ok = disc >= 0
                t = -b - np.sqrt(np.where(ok, disc, 0.0))
                upd = ok & (t > 1e-9) & (t < best)
                if upd.any():
                    best = np.where(upd, t, best)
                    p = o + best[:, None] * d
                    normal[upd] = ((p - c) / r)[upd]
                    sid[upd] = 16 + i
        return best, normal, sid

    def shade(self, o, d, rng_range, normal, sid):
        p = o + rng_range[:, None] * d
        l = self.light - p
        l /= np.linalg.norm(l, axis=1, keepdims=True)
        lam = np.maximum(0.0, (normal * l).sum(1))
        return self.albedo[sid] * (0.3 + 0.7 * lam)[:, None]

    def surface_distance(self, p):
        """Unsigned distance from points to the nearest surface (walls, boxes, spheres)."""
        dist = np.minimum(np.abs(p), np.abs(self.size - p)).min(axis=1)
        outside_room = np.any((p < 0) | (p > self.size), axis=1)
        dist = np.where(outside_room, np.linalg.norm(np.maximum(np.maximum(-p, p - self.size), 0.0),
                                                     axis=1), dist)
        for lo, hi in zip(self.box_lo, self.box_hi):
            q = np.maximum(np.maximum(lo - p, p - hi), 0.0)
            out = np.linalg.norm(q, axis=1)
            inn = np.minimum(p - lo, hi - p).min(axis=1)
            dist = np.minimum(dist, np.where(out > 0, out, np.abs(inn)))
        for c, r in zip(self.sph_c, self.sph_r):
            dist = np.minimum(dist, np.abs(np.linalg.norm(p - c, axis=1) - r))
        return dist


def near_surface_occupancy(room, G, extent, target_fraction):
    """bit = the cell centre is among the target_fraction of cells nearest to a surface (same distance as
    Room.surface_distance, evaluated on the whole grid with per-axis terms broadcast over [gz, gy, gx])."""
    ax = cell_centres_axis(G) * extent
    X, Y, Z = ax[None, None, :], ax[None, :, None], ax[:, None, None]
    axes = (X, Y, Z)
    sz = room.size
    # walls: inside the room the nearest wall; outside it the distance to the room box
    inside = [np.minimum(np.abs(a), np.abs(sz[i] - a)) for i, a in enumerate(axes)]
    outside = [np.maximum(np.maximum(-a, a - sz[i]), 0.0) for i, a in enumerate(axes)]
    d_in = np.minimum(np.minimum(inside[0], inside[1]), inside[2])
    d_out2 = outside[0] ** 2 + outside[1] ** 2 + outside[2] ** 2
    dist = np.where(d_out2 > 0, np.sqrt(d_out2), d_in)
    for lo, hi in zip(room.box_lo, room.box_hi):
        q = [np.maximum(np.maximum(lo[i] - a, a - hi[i]), 0.0) for i, a in enumerate(axes)]
        inn = [np.minimum(a - lo[i], hi[i] - a) for i, a in enumerate(axes)]
        out2 = q[0] ** 2 + q[1] ** 2 + q[2] ** 2
        d_inn = np.abs(np.minimum(np.minimum(inn[0], inn[1]), inn[2]))
        dist = np.minimum(dist, np.where(out2 > 0, np.sqrt(out2), d_inn))
    for c, r in zip(room.sph_c, room.sph_r):
        rr = np.sqrt((X - c[0]) ** 2 + (Y - c[1]) ** 2 + (Z - c[2]) ** 2)
        dist = np.minimum(dist, np.abs(rr - r))
    thr = np.quantile(dist.reshape(-1)[:: max(1, G ** 3 // (1 << 20))], target_fraction)
    mask = dist <= thr
    return pack_bits(mask.reshape(-1)), float(mask.mean())


def _mix64(x):
    """splitmix64 finaliser on uint64 arrays (input generation only: per-pixel random numbers that do not depend on
    which other pixels are evaluated)."""
    x = (x ^ (x >> np.uint64(30))) * np.uint64(0xbf58476d1ce4e5b9)
    x = (x ^ (x >> np.uint64(27))) * np.uint64(0x94d049bb133111eb)
    return x ^ (x >> np.uint64(31))


def pixel_uniform(seed, frame, pix, stream):
    """U[0,1) per (seed, frame, pixel, stream), counter-based."""
    with np.errstate(over="ignore"):
        k = _mix64(np.uint64(seed) * np.uint64(0x9e3779b97f4a7c15) + np.uint64(frame) * np.uint64(0xd1b54a32d192ed03) + np.uint64(stream))
        h = _mix64(k ^ (np.asarray(pix, np.uint64) * np.uint64(0x9e3779b97f4a7c15)))
    return (h >> np.uint64(11)).astype(np.float64) * 2.0 ** -53


class KeyframeSet:
    """n pinhole keyframes (fx=fy=600, cx=(W-1)/2, cy=(H-1)/2 at 1200x680; intrinsics scale with
    the resolution) with seeded look-at poses inside the room.  Per pixel: range r, RGB =
    albedo*(0.3+0.7 max(0,n.l)), D_slam = r(1+0.01 N(0,1)), Sigma_D = (0.01 r)^2; 5 % of pixels
    are outliers: D_slam = r U[0.3,2.0], Sigma_D = sigma_d^2, sigma_d ~ U[1,3].
    Whole frames are ray-cast lazily and cached; batches cast only the pixels they draw."""

    def __init__(self, room, seed, n, width=1200, height=680, outlier_fraction=0.05):
        self.room, self.seed, self.n, self.W, self.H = room, seed, n, width, height
        self.outlier_fraction = outlier_fraction      # BASELINE.json: 5 %; the ablation also runs heavier contamination
        s = width / 1200.0
        self.fx = self.fy = 600.0 * s
        self.cx, self.cy = (width - 1) / 2.0, (height - 1) / 2.0
        rng = np.random.Generator(np.random.PCG64([seed, 0xca3e]))
        self.centres, self.rot = [], []
        while len(self.centres) < n:
            c = 1.0 + rng.uniform(0, 1, 3) * (room.size - 2.0)
            tgt = rng.uniform(0, 1, 3) * room.size
            if room.inside_primitive(c[None])[0] or np.linalg.norm(tgt - c) < 0.5:
                continue
            f = (tgt - c) / np.linalg.norm(tgt - c)
            right = np.cross(f, np.array([0.0, 0.0, 1.0]))
            if np.linalg.norm(right) < 1e-3:
                continue
            right /= np.linalg.norm(right)
            down = np.cross(f, right)
            self.centres.append(c)
            self.rot.append(np.stack([right, down, f], axis=1))
        self._frames = {}

    def rays(self, i, pix=None):
        if pix is None:
            pix = np.arange(self.W * self.H)
        u, v = pix % self.W, pix // self.W
        dc = np.stack([(u - self.cx) / self.fx, (v - self.cy) / self.fy, np.ones(len(pix))], axis=1)
        dc /= np.linalg.norm(dc, axis=1, keepdims=True)
        d = dc @ self.rot[i].T
        o = np.broadcast_to(self.centres[i], d.shape).copy()
        return o, d

    def pixels(self, i, pix):
        """Keyframe i at the given pixel indices (ray cast on demand; every random number is a function of (seed, frame,
        pixel), so a pixel's values do not depend on which other pixels are asked for)."""
        pix = np.asarray(pix, np.int64)
        o, d = self.rays(i, pix)
        o32, d32 = o.astype(np.float32), d.astype(np.float32)      # cast what the field will see: the fp32 rays
        n = o.shape[0]
        r = np.empty(n)
        rgb = np.empty((n, 3))
        for a in range(0, n, 1 << 17):
            sl = slice(a, min(n, a + (1 << 17)))
            oo, dd = o32[sl].astype(np.float64), d32[sl].astype(np.float64)
            rr, nn, sid = self.room.cast(oo, dd)
            r[sl] = rr
            rgb[sl] = self.room.shade(oo, dd, rr, nn, sid)
        u = [pixel_uniform(self.seed, i, pix, k) for k in range(5)]
        gauss = np.sqrt(-2.0 * np.log(1.0 - u[0])) * np.cos(2.0 * np.pi * u[1])     # Box-Muller
        depth = r * (1.0 + 0.01 * gauss)
        var = (0.01 * r) ** 2
        outlier = u[2] < self.outlier_fraction
        depth = np.where(outlier, r * (0.3 + 1.7 * u[3]), depth)
        var = np.where(outlier, (1.0 + 2.0 * u[4]) ** 2, var)
        return dict(o=o32, d=d32, rgb=rgb.astype(np.float32), depth=depth.astype(np.float32), var=var.astype(np.float32),
                    range=r.astype(np.float32), outlier=outlier)

    def frame(self, i):
        if i not in self._frames:
            self._frames[i] = self.pixels(i, np.arange(self.W * self.H))
        return self._frames[i]

    def store_frame(self, i):
        """Keyframe i as a SLAM front end would hand it over: pinhole intrinsics, camera-to-world
        rotation and centre, image, z-DEPTH map and its variance (the ranges of frame() divided by |(xc, yc, 1)|,
        variances by its square)."""
        fr = self.frame(i)
        pix = np.arange(self.W * self.H)
        u, v = pix % self.W, pix // self.W
        n = np.sqrt(((u - self.cx) / self.fx) ** 2 + ((v - self.cy) / self.fy) ** 2 + 1.0)
        return dict(width=self.W, height=self.H, fx=self.fx, fy=self.fy, cx=self.cx, cy=self.cy,
                    R=self.rot[i].astype(np.float32), t=self.centres[i].astype(np.float32),
                    rgb=fr["rgb"].reshape(self.H, self.W, 3),
                    depth=(fr["depth"].astype(np.float64) / n).astype(np.float32).reshape(self.H, self.W),
                    depth_var=(fr["var"].astype(np.float64) / n ** 2).astype(np.float32).reshape(self.H, self.W))

    def draw_batch(self, step, R, t_min, t_max, K, batch_cls):
        rng = np.random.Generator(np.random.PCG64([self.seed, 0xba7c, step]))
        kf = rng.integers(0, self.n, R)
        pix = rng.integers(0, self.W * self.H, R)
        out = {k: np.empty((R, 3) if k in ("o", "d", "rgb") else (R,), np.float32)
               for k in ("o", "d", "rgb", "depth", "var")}
        for i in np.unique(kf):
            sel = kf == i
            if int(i) in self._frames:
                fr = {k: self._frames[int(i)][k][pix[sel]] for k in out}
            else:
                fr = self.pixels(int(i), pix[sel])
            for k in out:
                out[k][sel] = fr[k]
        return batch_cls(out["o"], out["d"], out["rgb"], out["depth"], out["var"], t_min, t_max, K)
