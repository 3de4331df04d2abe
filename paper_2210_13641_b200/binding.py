"""Thin Python binding of the C-ABI library (include/nsm.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of libnsm.so; this module only converts torch
device tensors to pointers.  PyTorch is used for device memory and streams.  There is no CPU
fallback: a missing or unloadable extension, or a missing GPU, raises.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnsm.so")

NSM_OK, NSM_ERR_INVALID_ARG, NSM_ERR_OOM, NSM_ERR_CUDA, NSM_ERR_CAPACITY, NSM_ERR_UNIMPLEMENTED = range(6)
NSM_MLP_FP32, NSM_MLP_FP16, NSM_MLP_BF16 = 0, 1, 2
NSM_OCC_FULL, NSM_OCC_SET, NSM_OCC_FROM_FIELD = 0, 1, 2
NSM_OPT_BATCH_READY, NSM_OPT_POSE_GRADIENTS, NSM_OPT_DEBUG_TIMELINE, NSM_OPT_POSE_LEVELS = 0, 1, 2, 3
NSM_MARCH_STATIC_MAX_RAYS = 1 << 20

DEBUG_ITEMS = dict(counts=(0, np.uint32), offsets=(1, np.uint32), s_ray=(2, np.uint32), s_k=(3, np.uint32),
                   s_t=(4, np.float32), s_delta=(5, np.float32), s_x=(6, np.float32), slots=(7, np.uint32),
                   w=(8, np.float32), e=(9, np.float32), sigma=(10, np.float32), rgb=(11, np.float32),
                   C=(12, np.float32), D_hat=(13, np.float32), O=(14, np.float32), dsigma=(15, np.float32),
                   drgb=(16, np.float32), grad=(17, np.float32), touched=(18, np.uint8),
                   hidden_density=(19, np.float32), hidden_color1=(20, np.float32), hidden_color2=(21, np.float32))

EXPORTS = ["nsm_create_field", "nsm_destroy_field", "nsm_update_occupancy", "nsm_get_occupancy",
           "nsm_train_step", "nsm_train_step_host", "nsm_backward", "nsm_apply_adam", "nsm_debug_set_grad",
           "nsm_render", "nsm_render_host", "nsm_param_count", "nsm_get_params", "nsm_set_params",
           "nsm_get_level_table", "nsm_debug_last_step", "nsm_total_samples", "nsm_profile", "nsm_set_option", "nsm_debug_timeline",
           "nsm_add_keyframe", "nsm_keyframe_count", "nsm_sample_batch", "nsm_train_step_sampled",
           "nsm_pose_gradients", "nsm_keyframe_pose_gradients", "nsm_apply_pose_step", "nsm_get_keyframe_pose",
           "nsm_update_occupancy_decay", "nsm_update_occupancy_stochastic", "nsm_get_occupancy_grid",
           "nsm_profile_read", "nsm_launch_count", "nsm_mlp_path", "nsm_march_static",
           "nsm_last_error", "nsm_version"]


class NsmFieldConfig(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("aabb_min", C.c_float * 3), ("aabb_extent", C.c_float),
                ("n_levels", C.c_uint32), ("n_features", C.c_uint32), ("log2_table_size", C.c_uint32),
                ("n_min", C.c_uint32), ("n_max", C.c_uint32), ("occ_res", C.c_uint32),
                ("density_hidden", C.c_uint32), ("density_out", C.c_uint32), ("geo_offset", C.c_uint32),
                ("geo_count", C.c_uint32), ("sh_degree", C.c_uint32), ("color_hidden", C.c_uint32),
                ("color_hidden_layers", C.c_uint32), ("mlp_precision", C.c_uint32), ("bg", C.c_float * 3),
                ("occ_sigma_threshold", C.c_float), ("lr", C.c_float), ("beta1", C.c_float),
                ("beta2", C.c_float), ("eps", C.c_float), ("sparse_table_adam", C.c_uint32),
                ("jitter", C.c_uint32), ("seed", C.c_uint64), ("max_rays", C.c_uint32),
                ("max_candidates", C.c_uint32), ("occ_cascades", C.c_uint32)]


class NsmRayBatch(C.Structure):
    _fields_ = [("n_rays", C.c_uint32), ("origins", C.c_void_p), ("dirs", C.c_void_p), ("rgb", C.c_void_p),
                ("depth", C.c_void_p), ("depth_var", C.c_void_p), ("t_min", C.c_float), ("t_max", C.c_float),
                ("n_candidates", C.c_uint32)]


class NsmKeyframeInfo(C.Structure):
    _fields_ = [("width", C.c_uint32), ("height", C.c_uint32), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("R", C.c_float * 9), ("t", C.c_float * 3)]


class NsmStepStats(C.Structure):
    _fields_ = [("loss", C.c_double), ("loss_rgb", C.c_double), ("loss_depth", C.c_double),
                ("n_samples", C.c_uint64), ("n_rays", C.c_uint32), ("step", C.c_uint32)]


class NsmMarchConfig(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("aabb_min", C.c_float * 3), ("aabb_extent", C.c_float),
                ("occ_res", C.c_uint32), ("occ_cascades", C.c_uint32), ("jitter", C.c_uint32), ("step", C.c_uint32),
                ("seed", C.c_uint64)]


class NsmMarchResult(C.Structure):
    _fields_ = [("capacity", C.c_uint64), ("counts", C.c_void_p), ("offsets", C.c_void_p), ("s_ray", C.c_void_p),
                ("s_k", C.c_void_p), ("s_t", C.c_void_p), ("s_delta", C.c_void_p), ("s_x", C.c_void_p)]


class NsmError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"nsm status {status}: {msg}")
        self.status = status


_LIB = None


def load_library():
    """Load libnsm.so (built in-tree by paper_2210_13641_b200/build.py).  Fails loudly if absent."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2210_13641_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, u64p, u32p = C.c_void_p, C.POINTER(C.c_uint64), C.POINTER(C.c_uint32)
        L.nsm_create_field.argtypes = [C.POINTER(NsmFieldConfig), vp, C.POINTER(vp)]
        L.nsm_destroy_field.argtypes = [vp]
        L.nsm_destroy_field.restype = None
        L.nsm_update_occupancy.argtypes = [vp, C.c_int, vp]
        L.nsm_get_occupancy.argtypes = [vp, vp]
        for name in ("nsm_train_step", "nsm_train_step_host", "nsm_backward"):
            getattr(L, name).argtypes = [vp, C.POINTER(NsmRayBatch), C.c_float, C.POINTER(NsmStepStats)]
        L.nsm_apply_adam.argtypes = [vp]
        L.nsm_debug_set_grad.argtypes = [vp, vp, vp]
        for name in ("nsm_render", "nsm_render_host"):
            getattr(L, name).argtypes = [vp, C.POINTER(NsmRayBatch), C.c_float, vp, vp, vp]
        L.nsm_param_count.argtypes = [vp, u64p, u64p]
        L.nsm_get_params.argtypes = [vp, vp, vp, vp, u32p]
        L.nsm_set_params.argtypes = [vp, vp, vp, vp, C.c_uint32]
        L.nsm_get_level_table.argtypes = [vp, u32p, u64p]
        L.nsm_debug_last_step.argtypes = [vp, C.c_int, vp, C.c_uint64, u64p]
        L.nsm_total_samples.argtypes = [vp, u64p]
        L.nsm_profile.argtypes = [vp, C.c_int]
        L.nsm_set_option.argtypes = [vp, C.c_int, C.c_uint32]
        L.nsm_pose_gradients.argtypes = [vp, vp, vp]
        L.nsm_keyframe_pose_gradients.argtypes = [vp, vp]
        L.nsm_update_occupancy_decay.argtypes = [vp, C.c_uint32, C.c_float]
        L.nsm_update_occupancy_stochastic.argtypes = [vp, C.c_uint32, C.c_float]
        L.nsm_get_occupancy_grid.argtypes = [vp, vp]
        L.nsm_apply_pose_step.argtypes = [vp, C.c_float, C.c_float]
        L.nsm_get_keyframe_pose.argtypes = [vp, C.c_uint32, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.nsm_add_keyframe.argtypes = [vp, C.POINTER(NsmKeyframeInfo), vp, vp, vp, u32p]
        L.nsm_keyframe_count.argtypes = [vp, u32p]
        L.nsm_sample_batch.argtypes = [vp, C.c_uint32, C.c_uint32, vp, vp, vp, vp, vp]
        L.nsm_train_step_sampled.argtypes = [vp, C.c_uint32, C.c_float, C.c_float, C.c_uint32, C.c_float, C.POINTER(NsmStepStats)]
        L.nsm_debug_timeline.argtypes = [vp, u64p, C.c_uint64, u32p]
        L.nsm_profile_read.argtypes = [vp, C.c_uint32, C.POINTER(C.c_char_p), C.POINTER(C.c_double), u64p, u32p]
        L.nsm_launch_count.argtypes = [vp]
        L.nsm_march_static.argtypes = [C.POINTER(NsmMarchConfig), C.POINTER(NsmRayBatch), vp, C.POINTER(NsmMarchResult), vp]
        L.nsm_launch_count.restype = C.c_uint64
        for name in ("nsm_mlp_path", "nsm_last_error", "nsm_version"):
            getattr(L, name).restype = C.c_char_p
        L.nsm_mlp_path.argtypes = [vp]
        _LIB = L
    return _LIB


def _check(status):
    if status != NSM_OK:
        raise NsmError(status, load_library().nsm_last_error().decode())


def make_config(fc):
    """fc: any object with the FieldConfig attribute names."""
    c = NsmFieldConfig()
    c.struct_size = C.sizeof(NsmFieldConfig)
    c.aabb_min[:] = [float(x) for x in fc.aabb_min]
    c.aabb_extent = float(fc.aabb_extent)
    for k in ("n_levels", "n_features", "log2_table_size", "n_min", "n_max", "occ_res", "density_hidden",
              "density_out", "geo_offset", "geo_count", "sh_degree", "color_hidden", "color_hidden_layers",
              "mlp_precision", "sparse_table_adam", "seed", "max_rays", "max_candidates"):
        setattr(c, k, int(getattr(fc, k)))
    c.jitter = int(getattr(fc, "jitter", 1))
    c.occ_cascades = int(getattr(fc, "occ_cascades", 1))
    c.bg[:] = [float(x) for x in fc.bg]
    for k in ("occ_sigma_threshold", "lr", "beta1", "beta2", "eps"):
        setattr(c, k, float(getattr(fc, k)))
    return c


def _dev_ptr(t, dtype=torch.float32):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous() and t.dtype == dtype, (t.device, t.dtype, t.is_contiguous())
    return t.data_ptr()


def _host_ptr(a):
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        assert not a.is_cuda and a.is_contiguous() and a.dtype == torch.float32
        return a.data_ptr()
    assert a.dtype == np.float32 and a.flags.c_contiguous
    return a.ctypes.data


class DeviceBatch:
    """A ray batch resident on the GPU (torch tensors keep the memory alive)."""

    def __init__(self, batch, device="cuda"):
        t = lambda a: None if a is None else torch.as_tensor(np.ascontiguousarray(a, np.float32)).to(device)
        self.origins, self.dirs = t(batch.origins), t(batch.dirs)
        self.rgb, self.depth, self.depth_var = t(batch.rgb), t(batch.depth), t(batch.depth_var)
        self.t_min, self.t_max, self.n_candidates = float(batch.t_min), float(batch.t_max), int(batch.n_candidates)
        self.n_rays = int(self.origins.shape[0])

    def c_struct(self):
        b = NsmRayBatch()
        b.n_rays = self.n_rays
        b.origins, b.dirs = _dev_ptr(self.origins), _dev_ptr(self.dirs)
        b.rgb, b.depth, b.depth_var = _dev_ptr(self.rgb), _dev_ptr(self.depth), _dev_ptr(self.depth_var)
        b.t_min, b.t_max, b.n_candidates = self.t_min, self.t_max, self.n_candidates
        return b


class MarchBuffers:
    """Caller-owned device arrays nsm_march_static writes (include/nsm.h nsm_march_result): allocated once, by torch,
    outside the call; capacity = samples per per-sample array."""

    def __init__(self, max_rays, capacity, device="cuda"):
        z = lambda n, dt: torch.zeros(n, dtype=dt, device=device)
        self.max_rays, self.capacity = int(max_rays), int(capacity)
        self.counts, self.offsets = z(self.max_rays, torch.int32), z(self.max_rays + 1, torch.int32)
        self.s_ray, self.s_k = z(self.capacity, torch.int32), z(self.capacity, torch.int32)
        self.s_t, self.s_delta = z(self.capacity, torch.float32), z(self.capacity, torch.float32)
        self.s_x = z(3 * self.capacity, torch.float32)

    def c_struct(self):
        r = NsmMarchResult()
        r.capacity = self.capacity
        for k in ("counts", "offsets", "s_ray", "s_k"):
            setattr(r, k, _dev_ptr(getattr(self, k), torch.int32))
        for k in ("s_t", "s_delta", "s_x"):
            setattr(r, k, _dev_ptr(getattr(self, k)))
        return r

    def read(self, n_rays):
        """The result of the last call as numpy arrays named like nsm_debug_last_step's items (synchronises)."""
        torch.cuda.synchronize(self.counts.device)
        u32 = lambda t, n: t[:n].cpu().numpy().view(np.uint32)
        offsets = u32(self.offsets, n_rays + 1)
        S = int(offsets[n_rays])
        return dict(counts=u32(self.counts, n_rays), offsets=offsets, s_ray=u32(self.s_ray, S), s_k=u32(self.s_k, S),
                    s_t=self.s_t[:S].cpu().numpy(), s_delta=self.s_delta[:S].cpu().numpy(),
                    s_x=self.s_x.view(3, self.capacity)[:, :S].t().contiguous().cpu().numpy())


def nsm_march_static(fc, batch, bits, out, step, stream=None):
    """S1-S3 alone through the entry point that allocates nothing (include/nsm.h).  fc: FieldConfig attribute names
    (aabb_min, aabb_extent, occ_res, occ_cascades, jitter, seed); batch: DeviceBatch; bits: uint8 device tensor or
    None (every cell live); out: MarchBuffers; step: the jitter stream's step index.  Enqueues and returns."""
    if not torch.cuda.is_available():
        raise RuntimeError("nsm needs a CUDA device (B200); there is no CPU fallback")
    lib = load_library()
    c = NsmMarchConfig()
    c.struct_size = C.sizeof(NsmMarchConfig)
    c.aabb_min[:] = [float(x) for x in fc.aabb_min]
    c.aabb_extent = float(fc.aabb_extent)
    c.occ_res, c.occ_cascades = int(fc.occ_res), int(getattr(fc, "occ_cascades", 1))
    c.jitter, c.step, c.seed = int(getattr(fc, "jitter", 1)), int(step), int(fc.seed)
    b, r = batch.c_struct(), out.c_struct()
    s = stream if stream is not None else torch.cuda.current_stream(out.counts.device)
    _check(lib.nsm_march_static(C.byref(c), C.byref(b), _dev_ptr(bits, torch.uint8), C.byref(r), C.c_void_p(s.cuda_stream)))


class HostBatch:
    """A ray batch in host memory for the *_host entry points: pinned (read in place by the kernels) or, with
    pinned=False, pageable (the library stages it with host-to-device copies)."""

    def __init__(self, batch, pinned=True):
        def pin(a):
            if a is None:
                return None
            t = torch.as_tensor(np.ascontiguousarray(a, np.float32))
            return t.pin_memory() if (pinned and torch.cuda.is_available()) else t
        self.origins, self.dirs = pin(batch.origins), pin(batch.dirs)
        self.rgb, self.depth, self.depth_var = pin(batch.rgb), pin(batch.depth), pin(batch.depth_var)
        self.t_min, self.t_max, self.n_candidates = float(batch.t_min), float(batch.t_max), int(batch.n_candidates)
        self.n_rays = int(self.origins.shape[0])

    def bytes_in(self):
        return sum(t.numel() * 4 for t in (self.origins, self.dirs, self.rgb, self.depth, self.depth_var) if t is not None)

    def c_struct(self):
        b = NsmRayBatch()
        b.n_rays = self.n_rays
        b.origins, b.dirs = _host_ptr(self.origins), _host_ptr(self.dirs)
        b.rgb, b.depth, b.depth_var = _host_ptr(self.rgb), _host_ptr(self.depth), _host_ptr(self.depth_var)
        b.t_min, b.t_max, b.n_candidates = self.t_min, self.t_max, self.n_candidates
        return b


def _stats(st):
    return dict(loss=st.loss, loss_rgb=st.loss_rgb, loss_depth=st.loss_depth, n_samples=int(st.n_samples),
                n_rays=int(st.n_rays), step=int(st.step))


class Field:
    """nsm_field handle.  Method names mirror the C entry points."""

    def __init__(self, fc, device="cuda:0", stream=None):
        if not torch.cuda.is_available():
            raise RuntimeError("nsm needs a CUDA device (B200); there is no CPU fallback")
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.fc = fc
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.cfg = make_config(fc)
        h = C.c_void_p()
        _check(self.lib.nsm_create_field(C.byref(self.cfg), C.c_void_p(self.stream.cuda_stream), C.byref(h)))
        self.h = h
        a, b = C.c_uint64(), C.c_uint64()
        _check(self.lib.nsm_param_count(self.h, C.byref(a), C.byref(b)))
        self.n_table, self.n_mlp = a.value, b.value
        res = (C.c_uint32 * fc.n_levels)()
        off = (C.c_uint64 * (fc.n_levels + 1))()
        _check(self.lib.nsm_get_level_table(self.h, res, off))
        self.res, self.offset = np.array(res, np.uint32), np.array(off, np.uint64)
        self.n_entries = int(self.offset[-1])

    def close(self):
        if getattr(self, "h", None):
            self.lib.nsm_destroy_field(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- parameters
    def mlp_shapes(self):
        fc = self.fc
        s = [("W_d1", fc.density_hidden, fc.n_levels * fc.n_features), ("W_d2", fc.density_out, fc.density_hidden),
             ("W_c1", fc.color_hidden, fc.geo_count + fc.sh_degree ** 2)]
        if fc.color_hidden_layers == 2:
            s.append(("W_c2", fc.color_hidden, fc.color_hidden))
        s.append(("W_c3", 3, fc.color_hidden))
        return s

    def nsm_set_params(self, theta=None, m=None, v=None, step=0):
        t = lambda a: None if a is None else torch.as_tensor(np.ascontiguousarray(a, np.float32)).to(self.device)
        th, mm, vv = t(theta), t(m), t(v)
        for a in (th, mm, vv):
            assert a is None or a.numel() == self.n_table + self.n_mlp
        _check(self.lib.nsm_set_params(self.h, _dev_ptr(th), _dev_ptr(mm), _dev_ptr(vv), int(step)))
        torch.cuda.synchronize(self.device)

    def nsm_get_params(self):
        P = self.n_table + self.n_mlp
        th, m, v = (torch.empty(P, dtype=torch.float32, device=self.device) for _ in range(3))
        step = C.c_uint32()
        _check(self.lib.nsm_get_params(self.h, _dev_ptr(th), _dev_ptr(m), _dev_ptr(v), C.byref(step)))
        torch.cuda.synchronize(self.device)
        return th.cpu().numpy(), m.cpu().numpy(), v.cpu().numpy(), step.value

    # ---- occupancy
    @property
    def n_occ_cells(self):
        """occ_cascades nested grids of occ_res^3 cells (marshalling: buffer sizes only)"""
        return max(int(getattr(self.fc, "occ_cascades", 1)), 1) * int(self.fc.occ_res) ** 3

    def nsm_update_occupancy(self, mode, bits=None, sync=True):
        d = None
        if bits is not None:
            d = torch.as_tensor(np.ascontiguousarray(bits, np.uint8)).to(self.device)
            assert d.numel() == (self.n_occ_cells + 7) // 8
            sync = True     # the staging tensor must outlive the copy
        _check(self.lib.nsm_update_occupancy(self.h, int(mode), _dev_ptr(d, torch.uint8)))
        if sync:
            torch.cuda.synchronize(self.device)

    def nsm_get_occupancy(self):
        d = torch.empty((self.n_occ_cells + 7) // 8, dtype=torch.uint8, device=self.device)
        _check(self.lib.nsm_get_occupancy(self.h, _dev_ptr(d, torch.uint8)))
        torch.cuda.synchronize(self.device)
        return d.cpu().numpy()

    # ---- steps
    def _step(self, fn, batch, lambda_d, want_stats):
        st = NsmStepStats()
        b = batch.c_struct()
        _check(fn(self.h, C.byref(b), float(lambda_d), C.byref(st) if want_stats else None))
        return _stats(st) if want_stats else None

    def nsm_train_step(self, batch, lambda_d, want_stats=True):
        return self._step(self.lib.nsm_train_step, batch, lambda_d, want_stats)

    def nsm_train_step_host(self, host_batch, lambda_d, want_stats=True):
        return self._step(self.lib.nsm_train_step_host, host_batch, lambda_d, want_stats)

    # ---- row F1: keyframe store and sampler
    def nsm_add_keyframe(self, kf):
        """kf: dict with width, height, fx, fy, cx, cy, R (3x3 camera-to-world), t (3,), rgb [H,W,3], depth [H,W]
        (z-depth), depth_var [H,W]; arrays may be numpy (uploaded here) or CUDA tensors.  Returns the keyframe index."""
        info = NsmKeyframeInfo()
        info.width, info.height = int(kf["width"]), int(kf["height"])
        info.fx, info.fy, info.cx, info.cy = (float(kf[n]) for n in ("fx", "fy", "cx", "cy"))
        info.R[:] = [float(x) for x in np.asarray(kf["R"], np.float32).reshape(9)]
        info.t[:] = [float(x) for x in np.asarray(kf["t"], np.float32).reshape(3)]
        dev = []
        for n in ("rgb", "depth", "depth_var"):
            a = kf[n]
            t = a if isinstance(a, torch.Tensor) else torch.as_tensor(np.ascontiguousarray(a, np.float32))
            dev.append(t.to(self.device, torch.float32).contiguous())
        idx = C.c_uint32()
        _check(self.lib.nsm_add_keyframe(self.h, C.byref(info), dev[0].data_ptr(), dev[1].data_ptr(), dev[2].data_ptr(), C.byref(idx)))
        torch.cuda.synchronize(self.device)      # the uploads above may be freed now
        return int(idx.value)

    def nsm_keyframe_count(self):
        n = C.c_uint32()
        _check(self.lib.nsm_keyframe_count(self.h, C.byref(n)))
        return int(n.value)

    def nsm_sample_batch(self, n_rays, draw):
        """Draw `draw` of n_rays rays as CUDA tensors: dict(origins, dirs, rgb, depth, depth_var)."""
        R = int(n_rays)
        out = dict(origins=torch.empty((R, 3), device=self.device), dirs=torch.empty((R, 3), device=self.device),
                   rgb=torch.empty((R, 3), device=self.device), depth=torch.empty(R, device=self.device),
                   depth_var=torch.empty(R, device=self.device))
        _check(self.lib.nsm_sample_batch(self.h, R, int(draw), *(out[k].data_ptr() for k in ("origins", "dirs", "rgb", "depth", "depth_var"))))
        return out

    def nsm_train_step_sampled(self, n_rays, t_min, t_max, n_candidates, lambda_d, want_stats=True):
        st = NsmStepStats()
        _check(self.lib.nsm_train_step_sampled(self.h, int(n_rays), float(t_min), float(t_max), int(n_candidates),
                                               float(lambda_d), C.byref(st) if want_stats else None))
        return _stats(st) if want_stats else None

    # ---- row f2: pose gradients
    def nsm_pose_gradients(self, n_rays):
        """(dL/do [R,3], rotation gradient d x dL/dd [R,3]) of the last step (needs NSM_OPT_POSE_GRADIENTS)."""
        go = torch.empty((int(n_rays), 3), device=self.device)
        tau = torch.empty((int(n_rays), 3), device=self.device)
        _check(self.lib.nsm_pose_gradients(self.h, go.data_ptr(), tau.data_ptr()))
        return go, tau

    def nsm_keyframe_pose_gradients(self):
        out = torch.empty((self.nsm_keyframe_count(), 6), device=self.device)
        _check(self.lib.nsm_keyframe_pose_gradients(self.h, out.data_ptr()))
        return out

    # ---- row f4: decayed partial occupancy refresh
    def nsm_update_occupancy_decay(self, n_subsets, decay, sync=True):
        _check(self.lib.nsm_update_occupancy_decay(self.h, int(n_subsets), float(decay)))
        if sync:
            torch.cuda.synchronize(self.device)

    def nsm_update_occupancy_stochastic(self, n_draws, decay, sync=True):
        _check(self.lib.nsm_update_occupancy_stochastic(self.h, int(n_draws), float(decay)))
        if sync:
            torch.cuda.synchronize(self.device)

    def nsm_get_occupancy_grid(self):
        out = torch.empty(self.n_occ_cells, device=self.device)
        _check(self.lib.nsm_get_occupancy_grid(self.h, out.data_ptr()))
        return out.cpu().numpy()

    def nsm_apply_pose_step(self, lr_translation, lr_rotation):
        _check(self.lib.nsm_apply_pose_step(self.h, float(lr_translation), float(lr_rotation)))

    def nsm_get_keyframe_pose(self, index):
        R, t = (C.c_float * 9)(), (C.c_float * 3)()
        _check(self.lib.nsm_get_keyframe_pose(self.h, int(index), R, t))
        return np.array(R, np.float32).reshape(3, 3), np.array(t, np.float32)

    def nsm_backward(self, batch, lambda_d, want_stats=True):
        return self._step(self.lib.nsm_backward, batch, lambda_d, want_stats)

    def nsm_apply_adam(self):
        _check(self.lib.nsm_apply_adam(self.h))

    def nsm_debug_set_grad(self, grad=None, touched=None):
        g = None if grad is None else torch.as_tensor(np.ascontiguousarray(grad, np.float32)).to(self.device)
        t = None if touched is None else torch.as_tensor(np.ascontiguousarray(touched, np.uint8)).to(self.device)
        _check(self.lib.nsm_debug_set_grad(self.h, _dev_ptr(g), _dev_ptr(t, torch.uint8)))
        torch.cuda.synchronize(self.device)

    def nsm_render(self, batch, cut=1e-4):
        R = batch.n_rays
        rgb = torch.empty((R, 3), dtype=torch.float32, device=self.device)
        depth = torch.empty(R, dtype=torch.float32, device=self.device)
        opac = torch.empty(R, dtype=torch.float32, device=self.device)
        b = batch.c_struct()
        _check(self.lib.nsm_render(self.h, C.byref(b), float(cut), _dev_ptr(rgb), _dev_ptr(depth), _dev_ptr(opac)))
        return rgb, depth, opac

    def nsm_render_host(self, host_batch, cut=1e-4, out=None):
        R = host_batch.n_rays
        if out is None:
            out = (torch.empty((R, 3), dtype=torch.float32).pin_memory(), torch.empty(R, dtype=torch.float32).pin_memory(),
                   torch.empty(R, dtype=torch.float32).pin_memory())
        b = host_batch.c_struct()
        _check(self.lib.nsm_render_host(self.h, C.byref(b), float(cut), out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr()))
        return out

    # ---- debug
    def nsm_debug_last_step(self, name):
        item, dt = DEBUG_ITEMS[name]
        n = C.c_uint64()
        _check(self.lib.nsm_debug_last_step(self.h, item, None, 0, C.byref(n)))
        buf = torch.empty(max(int(n.value), 1), dtype=torch.uint8, device=self.device)
        _check(self.lib.nsm_debug_last_step(self.h, item, buf.data_ptr(), n.value, None))
        torch.cuda.synchronize(self.device)
        a = buf[:n.value].cpu().numpy().view(dt)
        L, F = self.fc.n_levels, self.fc.n_features
        shape = dict(s_x=(-1, 3), slots=(-1, L, 8), w=(-1, L, 3), e=(-1, L * F), rgb=(-1, 3), C=(-1, 3), drgb=(-1, 3),
                     hidden_density=(-1, self.fc.density_hidden), hidden_color1=(-1, self.fc.color_hidden),
                     hidden_color2=(-1, self.fc.color_hidden))
        return a.reshape(shape[name]) if name in shape else a

    def nsm_total_samples(self):
        n = C.c_uint64()
        _check(self.lib.nsm_total_samples(self.h, C.byref(n)))
        return int(n.value)

    def nsm_debug_timeline(self):
        """[64, 2, n_kernels] uint64 globaltimer stamps (slot = step % 64); needs NSM_OPT_DEBUG_TIMELINE."""
        buf = (C.c_uint64 * (64 * 2 * 32))()
        nk = C.c_uint32()
        _check(self.lib.nsm_debug_timeline(self.h, buf, 64 * 2 * 32, C.byref(nk)))
        return np.frombuffer(buf, np.uint64)[:64 * 2 * nk.value].reshape(64, 2, nk.value).copy()

    def nsm_set_option(self, opt, value):
        _check(self.lib.nsm_set_option(self.h, int(opt), int(value)))

    def nsm_profile(self, enable):
        _check(self.lib.nsm_profile(self.h, int(bool(enable))))

    def nsm_profile_read(self):
        """{kernel class: (total ms, launches)} since nsm_profile(True)."""
        cap = 32
        names = (C.c_char_p * cap)()
        ms = (C.c_double * cap)()
        cnt = (C.c_uint64 * cap)()
        n = C.c_uint32()
        _check(self.lib.nsm_profile_read(self.h, cap, names, ms, cnt, C.byref(n)))
        return {names[i].decode(): (ms[i], int(cnt[i])) for i in range(n.value)}

    def nsm_launch_count(self):
        return int(self.lib.nsm_launch_count(self.h))

    def nsm_mlp_path(self):
        return self.lib.nsm_mlp_path(self.h).decode()
