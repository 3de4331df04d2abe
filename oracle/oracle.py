"""ctypes binding of the float64 CPU oracle (oracle/nsm_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It does not import, and is not imported by, the CUDA package.  Argument
marshalling only: all arithmetic is in nsm_oracle.c.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
_f32p, _f64p, _u32p, _u8p, _u64p = (C.POINTER(t) for t in
                                    (C.c_float, C.c_double, C.c_uint32, C.c_uint8, C.c_uint64))


class OrcConfig(C.Structure):
    _fields_ = [("aabb_min", C.c_float * 3), ("aabb_extent", C.c_float),
                ("n_levels", C.c_uint32), ("n_features", C.c_uint32),
                ("log2_table_size", C.c_uint32), ("n_min", C.c_uint32), ("n_max", C.c_uint32),
                ("occ_res", C.c_uint32), ("density_hidden", C.c_uint32),
                ("density_out", C.c_uint32), ("geo_offset", C.c_uint32),
                ("geo_count", C.c_uint32), ("sh_degree", C.c_uint32),
                ("color_hidden", C.c_uint32), ("color_hidden_layers", C.c_uint32),
                ("bg", C.c_float * 3), ("occ_sigma_threshold", C.c_float),
                ("lr", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float),
                ("sparse_table_adam", C.c_uint32), ("seed", C.c_uint64), ("occ_cascades", C.c_uint32),
                ("pose_levels", C.c_uint32)]


class OrcBatch(C.Structure):
    _fields_ = [("n_rays", C.c_uint32), ("origins", _f32p), ("dirs", _f32p), ("rgb", _f32p),
                ("depth", _f32p), ("depth_var", _f32p), ("t_min", C.c_float), ("t_max", C.c_float),
                ("n_candidates", C.c_uint32)]


class OrcKeyframe(C.Structure):
    _fields_ = [("width", C.c_uint32), ("height", C.c_uint32), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("R", C.c_float * 9), ("t", C.c_float * 3),
                ("rgb", C.POINTER(C.c_float)), ("depth", C.POINTER(C.c_float)), ("depth_var", C.POINTER(C.c_float))]


class OrcStats(C.Structure):
    _fields_ = [("loss", C.c_double), ("loss_rgb", C.c_double), ("loss_depth", C.c_double),
                ("n_samples", C.c_uint64), ("n_rays", C.c_uint32), ("step", C.c_uint32)]


class OrcTrace(C.Structure):
    _fields_ = [("counts", _u32p), ("offsets", _u32p), ("s_ray", _u32p), ("s_k", _u32p),
                ("s_t", _f32p), ("s_delta", _f32p), ("s_x", _f32p), ("slots", _u32p), ("w", _f32p),
                ("e", _f64p), ("sigma", _f64p), ("rgb", _f64p), ("C", _f64p), ("D_hat", _f64p),
                ("O", _f64p), ("dsigma", _f64p), ("drgb", _f64p), ("grad", _f64p),
                ("touched", _u8p), ("g_o", _f64p), ("tau", _f64p), ("dx", _f64p)]


_LIBS = {}


def lib(omp=False):
    """Load (building if stale) the oracle shared object."""
    key = bool(omp)
    if key not in _LIBS:
        outs = _build.build()
        L = C.CDLL(outs["libnsm_oracle_omp.so" if omp else "libnsm_oracle.so"])
        L.orc_level_table.argtypes = [C.POINTER(OrcConfig), _u32p, _u64p]
        L.orc_param_count.argtypes = [C.POINTER(OrcConfig), _u64p, _u64p]
        L.orc_mlp_offsets.argtypes = [C.POINTER(OrcConfig), _u64p]
        L.orc_hash32.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]
        L.orc_hash32.restype = C.c_uint32
        L.orc_jitter_u.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]
        L.orc_jitter_u.restype = C.c_float
        L.orc_march.argtypes = [C.POINTER(OrcConfig), _u8p, C.POINTER(OrcBatch), C.c_int,
                                C.c_uint32, _u32p, _u32p, _u32p, _u32p, _f32p, _f32p, _f32p]
        L.orc_march.restype = C.c_int64
        L.orc_encode.argtypes = [C.POINTER(OrcConfig), _f64p, C.c_uint64, _f32p, _u32p, _f32p, _f64p]
        L.orc_sh.argtypes = [C.c_uint32, _f64p, _f64p]
        L.orc_sh.restype = None
        L.orc_field_eval.argtypes = [C.POINTER(OrcConfig), _f64p, _f64p, _f64p, _f64p, _f64p]
        L.orc_composite.argtypes = [C.c_uint32, _f64p, _f64p, _f32p, _f32p, _f32p, C.c_double,
                                    _f64p, _f64p, _f64p]
        L.orc_composite.restype = None
        L.orc_train_step.argtypes = [C.POINTER(OrcConfig), _f64p, _f64p, _f64p, _u32p, _u8p,
                                     C.POINTER(OrcBatch), C.c_double, C.c_int, C.c_int,
                                     C.POINTER(OrcStats), C.POINTER(OrcTrace)]
        L.orc_adam.argtypes = [C.c_uint64, _f64p, _f64p, _f64p, _f64p, _u8p, C.c_uint32, C.c_uint32,
                               C.c_double, C.c_double, C.c_double, C.c_double]
        L.orc_adam.restype = None
        L.orc_occupancy_from_field.argtypes = [C.POINTER(OrcConfig), _f64p, _u8p, _f64p]
        L.orc_render.argtypes = [C.POINTER(OrcConfig), _f64p, _u8p, C.POINTER(OrcBatch), C.c_double,
                                 _f64p, _f64p, _f64p, _u64p]
        L.orc_sample_batch.argtypes = [C.POINTER(OrcKeyframe), C.c_uint32, C.c_uint64, C.c_uint32, C.c_uint32,
                                       _u32p, _u32p, _f32p, _f32p, _f32p, _f32p, _f32p]
        L.orc_sample_batch.restype = None
        L.orc_occupancy_decay_update.argtypes = [C.POINTER(OrcConfig), _f64p, _f64p, C.c_uint32, C.c_uint32, C.c_double,
                                                 _u8p, _f64p]
        L.orc_occupancy_stochastic_update.argtypes = [C.POINTER(OrcConfig), _f64p, _f64p, C.c_uint32, C.c_uint32, C.c_double,
                                                      _u8p, _u64p, _f32p, _f64p]
        L.orc_occupancy_cell.argtypes = [C.POINTER(OrcConfig), _f32p, _u32p]
        L.orc_occupancy_cell.restype = C.c_uint64
        L.orc_occupancy_cell_point.argtypes = [C.POINTER(OrcConfig), C.c_uint64, _f32p, _f32p]
        L.orc_occupancy_cell_point.restype = None
        L.orc_pose_step.argtypes = [_f64p, _f64p, _f64p, _f64p, _u32p, _f64p, C.c_double, C.c_double, C.c_double,
                                    C.c_double, C.c_double]
        L.orc_pose_step.restype = None
        L.orc_num_threads.restype = C.c_int
        _LIBS[key] = L
    return _LIBS[key]


def _p(a, typ):
    return None if a is None else a.ctypes.data_as(typ)


def make_config(fc):
    """fc: any object with the FieldConfig attribute names (workloads.configs.FieldConfig)."""
    c = OrcConfig()
    c.aabb_min[:] = [float(x) for x in fc.aabb_min]
    c.aabb_extent = float(fc.aabb_extent)
    for k in ("n_levels", "n_features", "log2_table_size", "n_min", "n_max", "occ_res",
              "density_hidden", "density_out", "geo_offset", "geo_count", "sh_degree",
              "color_hidden", "color_hidden_layers", "sparse_table_adam", "seed"):
        setattr(c, k, int(getattr(fc, k)))
    c.bg[:] = [float(x) for x in fc.bg]
    for k in ("occ_sigma_threshold", "lr", "beta1", "beta2", "eps"):
        setattr(c, k, float(getattr(fc, k)))
    c.occ_cascades = int(getattr(fc, "occ_cascades", 1))
    c.pose_levels = int(getattr(fc, "pose_levels", 0))
    return c


def n_occ_cells(fc):
    """Cells of the occupancy structure: occ_cascades grids of occ_res^3 (F4 / R23)."""
    return max(int(getattr(fc, "occ_cascades", 1)), 1) * int(fc.occ_res) ** 3


def occupancy_cell(fc, x):
    """R23: (bit index, cascade) of the occupancy cell that tests the normalised positions x [n,3]."""
    c = make_config(fc)
    x = np.ascontiguousarray(x, np.float32).reshape(-1, 3)
    cell = np.empty(len(x), np.uint64)
    casc = np.empty(len(x), np.uint32)
    L, j = lib(), C.c_uint32()
    for i in range(len(x)):
        cell[i] = L.orc_occupancy_cell(C.byref(c), _p(x[i], _f32p), C.byref(j))
        casc[i] = j.value
    return cell, casc


def occupancy_cell_point(fc, cells, u=None):
    """The normalised positions of the points at offsets u [n,3] (default: the centres) inside the given cells."""
    c = make_config(fc)
    cells = np.asarray(cells, np.uint64).reshape(-1)
    u = np.full((len(cells), 3), 0.5, np.float32) if u is None else np.ascontiguousarray(u, np.float32).reshape(-1, 3)
    out = np.empty((len(cells), 3), np.float32)
    L = lib()
    for i in range(len(cells)):
        L.orc_occupancy_cell_point(C.byref(c), int(cells[i]), _p(u[i], _f32p), _p(out[i], _f32p))
    return out


class _BatchHolder:
    """Keeps the contiguous fp32 arrays alive for the duration of a call."""

    def __init__(self, batch):
        f = lambda a: None if a is None else np.ascontiguousarray(a, dtype=np.float32)
        self.o, self.d = f(batch.origins), f(batch.dirs)
        self.rgb, self.depth, self.var = f(batch.rgb), f(batch.depth), f(batch.depth_var)
        b = OrcBatch()
        b.n_rays = int(self.o.shape[0])
        b.origins, b.dirs = _p(self.o, _f32p), _p(self.d, _f32p)
        b.rgb, b.depth, b.depth_var = _p(self.rgb, _f32p), _p(self.depth, _f32p), _p(self.var, _f32p)
        b.t_min, b.t_max = float(np.float32(batch.t_min)), float(np.float32(batch.t_max))
        b.n_candidates = int(batch.n_candidates)
        self.c = b


def level_table(fc):
    c = make_config(fc)
    res = np.zeros(fc.n_levels, np.uint32)
    off = np.zeros(fc.n_levels + 1, np.uint64)
    if lib().orc_level_table(C.byref(c), _p(res, _u32p), _p(off, _u64p)) != 0:
        raise ValueError("bad level configuration")
    return res, off


def param_count(fc):
    c = make_config(fc)
    a, b = C.c_uint64(), C.c_uint64()
    if lib().orc_param_count(C.byref(c), C.byref(a), C.byref(b)) != 0:
        raise ValueError("bad configuration")
    return a.value, b.value


def mlp_offsets(fc):
    c = make_config(fc)
    out = np.zeros(fc.color_hidden_layers + 4, np.uint64)
    if lib().orc_mlp_offsets(C.byref(c), _p(out, _u64p)) != 0:
        raise ValueError("bad configuration")
    return out


def mlp_shapes(fc):
    """[(name, n_out, n_in)] in canonical order."""
    lf = fc.n_levels * fc.n_features
    ci = fc.geo_count + fc.sh_degree ** 2
    s = [("W_d1", fc.density_hidden, lf), ("W_d2", fc.density_out, fc.density_hidden),
         ("W_c1", fc.color_hidden, ci)]
    if fc.color_hidden_layers == 2:
        s.append(("W_c2", fc.color_hidden, fc.color_hidden))
    s.append(("W_c3", 3, fc.color_hidden))
    return s


def hash32(seed, step, r, k):
    return int(lib().orc_hash32(seed, step, r, k))


def jitter_u(seed, step, r, k):
    return float(lib().orc_jitter_u(seed, step, r, k))


def march(fc, bits, batch, jitter=True, step=1):
    c = make_config(fc)
    h = _BatchHolder(batch)
    R, K = h.c.n_rays, h.c.n_candidates
    cap = R * K
    out = dict(counts=np.zeros(R, np.uint32), offsets=np.zeros(R + 1, np.uint32),
               s_ray=np.zeros(cap, np.uint32), s_k=np.zeros(cap, np.uint32),
               s_t=np.zeros(cap, np.float32), s_delta=np.zeros(cap, np.float32),
               s_x=np.zeros((cap, 3), np.float32))
    bits = None if bits is None else np.ascontiguousarray(bits, np.uint8)
    S = lib().orc_march(C.byref(c), _p(bits, _u8p), C.byref(h.c), int(bool(jitter)), int(step),
                        _p(out["counts"], _u32p), _p(out["offsets"], _u32p),
                        _p(out["s_ray"], _u32p), _p(out["s_k"], _u32p), _p(out["s_t"], _f32p),
                        _p(out["s_delta"], _f32p), _p(out["s_x"], _f32p))
    if S < 0:
        raise ValueError("orc_march failed")
    for k in ("s_ray", "s_k", "s_t", "s_delta", "s_x"):
        out[k] = out[k][:S]
    out["S"] = int(S)
    return out


def encode(fc, theta, x, want_index=True):
    c = make_config(fc)
    x = np.ascontiguousarray(x, np.float32).reshape(-1, 3)
    theta = np.ascontiguousarray(theta, np.float64)
    S, L, F = x.shape[0], fc.n_levels, fc.n_features
    e = np.zeros((S, L * F), np.float64)
    slots = np.zeros((S, L, 8), np.uint32) if want_index else None
    w = np.zeros((S, L, 3), np.float32) if want_index else None
    if lib().orc_encode(C.byref(c), _p(theta, _f64p), S, _p(x, _f32p), _p(slots, _u32p),
                        _p(w, _f32p), _p(e, _f64p)) != 0:
        raise ValueError("orc_encode failed")
    return e, slots, w


def sh(n, d):
    d = np.ascontiguousarray(d, np.float64).reshape(-1, 3)
    Y = np.zeros((d.shape[0], n * n), np.float64)
    L = lib()
    for i in range(d.shape[0]):
        L.orc_sh(n, _p(d[i], _f64p), _p(Y[i], _f64p))
    return Y


def field_eval(fc, theta_mlp, e, Y):
    c = make_config(fc)
    theta_mlp = np.ascontiguousarray(theta_mlp, np.float64)
    e = np.ascontiguousarray(e, np.float64)
    Y = np.ascontiguousarray(Y, np.float64)
    sig = C.c_double()
    rgb = np.zeros(3, np.float64)
    if lib().orc_field_eval(C.byref(c), _p(theta_mlp, _f64p), _p(e, _f64p), _p(Y, _f64p),
                            C.byref(sig), _p(rgb, _f64p)) != 0:
        raise ValueError("orc_field_eval failed")
    return sig.value, rgb


def composite(sigma, rgb, t, delta, bg=(0, 0, 0), cut=0.0):
    sigma = np.ascontiguousarray(sigma, np.float64)
    rgb = np.ascontiguousarray(rgb, np.float64).reshape(-1, 3)
    t = np.ascontiguousarray(t, np.float32)
    delta = np.ascontiguousarray(delta, np.float32)
    bg = np.ascontiguousarray(bg, np.float32)
    Cc = np.zeros(3, np.float64)
    D, O = C.c_double(), C.c_double()
    lib().orc_composite(len(sigma), _p(sigma, _f64p), _p(rgb, _f64p), _p(t, _f32p),
                        _p(delta, _f32p), _p(bg, _f32p), float(cut), _p(Cc, _f64p), C.byref(D),
                        C.byref(O))
    return Cc, D.value, O.value


def adam(theta, m, v, g, step, lr, beta1, beta2, eps, mask=None, mask_group=1):
    for a in (theta, m, v):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    g = np.ascontiguousarray(g, np.float64)
    mask = None if mask is None else np.ascontiguousarray(mask, np.uint8)
    lib().orc_adam(theta.size, _p(theta, _f64p), _p(m, _f64p), _p(v, _f64p), _p(g, _f64p),
                   _p(mask, _u8p), int(mask_group), int(step), lr, beta1, beta2, eps)


def sample_batch(keyframes, seed, draw, n_rays):
    """F1: the ray-batch sampler.  keyframes: list of dicts with width, height, fx, fy, cx, cy, R (3x3 camera-to-world),
    t (3,), rgb [H,W,3], depth [H,W] (z-depth), depth_var [H,W].  Returns a dict of arrays (kf, pix, origins, dirs,
    rgb, depth, depth_var)."""
    arr = (OrcKeyframe * len(keyframes))()
    keep = []
    for a, k in zip(arr, keyframes):
        a.width, a.height = int(k["width"]), int(k["height"])
        a.fx, a.fy, a.cx, a.cy = (float(np.float32(k[n])) for n in ("fx", "fy", "cx", "cy"))
        a.R[:] = [float(x) for x in np.asarray(k["R"], np.float32).reshape(9)]
        a.t[:] = [float(x) for x in np.asarray(k["t"], np.float32).reshape(3)]
        bufs = [np.ascontiguousarray(k[n], np.float32).reshape(-1) for n in ("rgb", "depth", "depth_var")]
        assert bufs[0].size == 3 * a.width * a.height and bufs[1].size == bufs[2].size == a.width * a.height
        keep.append(bufs)
        a.rgb, a.depth, a.depth_var = (_p(b, _f32p) for b in bufs)
    R = int(n_rays)
    out = dict(kf=np.empty(R, np.uint32), pix=np.empty(R, np.uint32), origins=np.empty((R, 3), np.float32),
               dirs=np.empty((R, 3), np.float32), rgb=np.empty((R, 3), np.float32), depth=np.empty(R, np.float32),
               depth_var=np.empty(R, np.float32))
    lib().orc_sample_batch(arr, len(keyframes), int(seed), int(draw), R, _p(out["kf"], _u32p), _p(out["pix"], _u32p),
                           _p(out["origins"], _f32p), _p(out["dirs"], _f32p), _p(out["rgb"], _f32p),
                           _p(out["depth"], _f32p), _p(out["depth_var"], _f32p))
    return out


def pose_step(R, t, m, v, count, g, lr_t, lr_r, beta1=0.9, beta2=0.99, eps=1e-15):
    """F2 update of one keyframe, in place on float64 arrays R (3,3), t (3,), m (6,), v (6,); returns the new count."""
    for a in (R, t, m, v):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    cnt = np.array([count], np.uint32)
    g = np.ascontiguousarray(g, np.float64)
    lib().orc_pose_step(_p(R, _f64p), _p(t, _f64p), _p(m, _f64p), _p(v, _f64p), _p(cnt, _u32p), _p(g, _f64p),
                        float(lr_t), float(lr_r), float(beta1), float(beta2), float(eps))
    return int(cnt[0])


class Oracle:
    """A field's float64 state (theta, m, v, step, occupancy bits) plus the oracle's steps."""

    def __init__(self, fc, theta0, omp=False):
        self.fc = fc
        self.cfg = make_config(fc)
        self.lib = lib(omp)
        self.n_table, self.n_mlp = param_count(fc)
        self.res, self.offset = level_table(fc)
        self.n_entries = int(self.offset[-1])
        P = self.n_table + self.n_mlp
        theta0 = np.asarray(theta0)
        assert theta0.shape == (P,), (theta0.shape, P)
        self.theta = theta0.astype(np.float64)
        self.m = np.zeros(P, np.float64)
        self.v = np.zeros(P, np.float64)
        self.step = 0
        self.bits = None  # None == FULL

    def set_occupancy(self, bits):
        self.bits = None if bits is None else np.ascontiguousarray(bits, np.uint8).copy()

    def occupancy_from_field(self, want_sigma=False):
        n = n_occ_cells(self.fc)
        bits = np.zeros((n + 7) // 8, np.uint8)
        sig = np.zeros(n, np.float64) if want_sigma else None
        if self.lib.orc_occupancy_from_field(C.byref(self.cfg), _p(self.theta, _f64p),
                                             _p(bits, _u8p), _p(sig, _f64p)) != 0:
            raise ValueError("orc_occupancy_from_field failed")
        self.bits = bits
        if sig is not None:
            self.occ_grid, self.occ_updates = sig.copy(), 0     # F4: a full refresh seeds the running grid
        return (bits, sig) if want_sigma else bits

    def occupancy_decay_update(self, n_sub, decay, want_sigma=False):
        """F4: decayed running-maximum grid with a strided 1/n_sub refresh; keeps self.occ_grid and self.occ_updates."""
        n = n_occ_cells(self.fc)
        if getattr(self, "occ_grid", None) is None:
            self.occ_grid, self.occ_updates = np.zeros(n, np.float64), 0
        bits = np.zeros((n + 7) // 8, np.uint8)
        vis = np.zeros(n, np.float64) if want_sigma else None
        if self.lib.orc_occupancy_decay_update(C.byref(self.cfg), _p(self.theta, _f64p), _p(self.occ_grid, _f64p),
                                               self.occ_updates, int(n_sub), float(decay), _p(bits, _u8p), _p(vis, _f64p)) != 0:
            raise ValueError("orc_occupancy_decay_update failed")
        self.occ_updates += 1
        self.bits = bits
        return (bits, vis) if want_sigma else bits

    def occupancy_stochastic_update(self, n_draws, decay, want_draws=False):
        """F4 (R25): decayed running-maximum grid refreshed at n_draws random points; self.occ_draws counts these updates
        (it keys the draws and is never reset)."""
        n = n_occ_cells(self.fc)
        if getattr(self, "occ_grid", None) is None:
            self.occ_grid, self.occ_updates = np.zeros(n, np.float64), 0
        self.occ_draws = getattr(self, "occ_draws", 0)
        bits = np.zeros((n + 7) // 8, np.uint8)
        cells = np.zeros(n_draws, np.uint64) if want_draws else None
        x = np.zeros((n_draws, 3), np.float32) if want_draws else None
        sig = np.zeros(n_draws, np.float64) if want_draws else None
        if self.lib.orc_occupancy_stochastic_update(C.byref(self.cfg), _p(self.theta, _f64p), _p(self.occ_grid, _f64p),
                                                    self.occ_draws, int(n_draws), float(decay), _p(bits, _u8p),
                                                    _p(cells, _u64p), _p(x, _f32p), _p(sig, _f64p)) != 0:
            raise ValueError("orc_occupancy_stochastic_update failed")
        self.occ_draws += 1
        self.bits = bits
        return (bits, cells, x, sig) if want_draws else bits

    def train_step(self, batch, lambda_d, jitter=True, apply_adam=True, trace=(), ):
        """trace: iterable of OrcTrace field names to return.  Returns (stats dict, trace dict)."""
        h = _BatchHolder(batch)
        R, K = h.c.n_rays, h.c.n_candidates
        cap, L, F = R * K, self.fc.n_levels, self.fc.n_features
        P = self.n_table + self.n_mlp
        shapes = dict(counts=((R,), np.uint32), offsets=((R + 1,), np.uint32),
                      s_ray=((cap,), np.uint32), s_k=((cap,), np.uint32),
                      s_t=((cap,), np.float32), s_delta=((cap,), np.float32),
                      s_x=((cap, 3), np.float32), slots=((cap, L, 8), np.uint32),
                      w=((cap, L, 3), np.float32), e=((cap, L * F), np.float64),
                      sigma=((cap,), np.float64), rgb=((cap, 3), np.float64),
                      C=((R, 3), np.float64), D_hat=((R,), np.float64), O=((R,), np.float64),
                      dsigma=((cap,), np.float64), drgb=((cap, 3), np.float64),
                      grad=((P,), np.float64), touched=((self.n_entries,), np.uint8),
                      g_o=((R, 3), np.float64), tau=((R, 3), np.float64), dx=((cap, 3), np.float64))
        tr = OrcTrace()
        out = {}
        for name in trace:
            shp, dt = shapes[name]
            out[name] = np.zeros(shp, dt)
            typ = dict(OrcTrace._fields_)[name]
            setattr(tr, name, out[name].ctypes.data_as(typ))
        st = OrcStats()
        step = C.c_uint32(self.step)
        rc = self.lib.orc_train_step(C.byref(self.cfg), _p(self.theta, _f64p), _p(self.m, _f64p),
                                     _p(self.v, _f64p), C.byref(step), _p(self.bits, _u8p),
                                     C.byref(h.c), float(lambda_d), int(bool(jitter)),
                                     int(bool(apply_adam)), C.byref(st), C.byref(tr))
        if rc != 0:
            raise RuntimeError(f"orc_train_step failed ({rc})")
        self.step = step.value
        S = int(st.n_samples)
        for name in out:
            if shapes[name][0][0] == cap:
                out[name] = out[name][:S]
        stats = dict(loss=st.loss, loss_rgb=st.loss_rgb, loss_depth=st.loss_depth, n_samples=S,
                     n_rays=int(st.n_rays), step=int(st.step))
        return stats, out

    def render(self, batch, cut=1e-4):
        h = _BatchHolder(batch)
        R = h.c.n_rays
        rgb = np.zeros((R, 3), np.float64)
        depth = np.zeros(R, np.float64)
        opac = np.zeros(R, np.float64)
        n = C.c_uint64()
        if self.lib.orc_render(C.byref(self.cfg), _p(self.theta, _f64p), _p(self.bits, _u8p),
                               C.byref(h.c), float(cut), _p(rgb, _f64p), _p(depth, _f64p),
                               _p(opac, _f64p), C.byref(n)) != 0:
            raise RuntimeError("orc_render failed")
        return rgb, depth, opac, int(n.value)

    def num_threads(self):
        return int(self.lib.orc_num_threads())
