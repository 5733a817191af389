"""Thin ctypes binding of ``libsplx.so`` (C ABI: ``include/splx.h``) -- argument marshalling only.

Every function has the name of the C entry point without the ``splx_`` prefix and takes torch
CUDA tensors (PyTorch is used for device memory and streams only); every step of the path
runs in the CUDA kernels behind the ABI.  There is no CPU fallback: if ``libsplx.so`` is
missing or no CUDA device is present, the first call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsplx.so")
_lib = None

G2D_STRIDE = 12
BLEND_STRIDE = 12
TILE = 16
MAX_K = 64
PB_CLEAR_G2D, PB_OVERWRITE = 1, 2
OK, ERR_INVALID_ARG, ERR_WORKSPACE, ERR_CAPACITY, ERR_CUDA = 0, -1, -2, -3, -4

EXPORTS = [
    "splx_create", "splx_destroy", "splx_last_error", "splx_set_stream", "splx_launch_count",
    "splx_slot_map_words", "splx_slot_map",
    "splx_project", "splx_bin_sort_ws_bytes", "splx_bin_sort", "splx_check_capacity",
    "splx_render_partial", "splx_compose", "splx_l1_loss_grad", "splx_compose_backward",
    "splx_raster_backward", "splx_project_backward", "splx_backward_ws_bytes", "splx_backward",
    "splx_adam", "splx_adam_groups",
    "splx_visible_regions", "splx_schedule_views", "splx_project_plan", "splx_project_geometry_plan",
    "splx_project_colour_list_plan", "splx_bin_sort_plan",
    "splx_render_partial_plan", "splx_compose_plan", "splx_compose_backward_plan",
    "splx_raster_backward_plan", "splx_project_backward_plan", "splx_backward_plan",
    "splx_compose_l1_backward_plan",
    "splx_bin_sort_visible", "splx_bin_sort_gradient_rows", "splx_project_backward_list_plan", "splx_adam_sparse",
    "splx_cross_sets", "splx_cross_depth_ranges", "splx_bin_sort_filtered_plan",
    "splx_adam_groups_flagged", "splx_dssim_ws_floats", "splx_dssim_loss_grad", "splx_dssim_loss_grad_static", "splx_iteration", "splx_microbench",
]
MAX_VIEWS = 8
DSSIM_STATIC_MAX_PIXELS = 262144
TILE_INVISIBLE, TILE_SATURATED = 1, 2
PLAN_SPARSE = 1
ORDER_EXTRA = 1025


class SplxError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libsplx error {code}: {msg}")
        self.code = code


class Config(C.Structure):
    _fields_ = [("alpha_min", C.c_float), ("alpha_max", C.c_float), ("T_eps", C.c_float),
                ("dilation", C.c_float), ("lim_factor", C.c_float), ("radius_floor", C.c_float)]


class CameraS(C.Structure):
    _fields_ = [("R", C.c_float * 9), ("t", C.c_float * 3), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("width", C.c_int32), ("height", C.c_int32),
                ("near_z", C.c_float)]


class GaussiansS(C.Structure):
    _fields_ = [("mean", C.c_void_p), ("log_scale", C.c_void_p), ("quat", C.c_void_p),
                ("opacity_logit", C.c_void_p), ("sh", C.c_void_p), ("n", C.c_int64)]


class ProjectedS(C.Structure):
    _fields_ = [("means2d", C.c_void_p), ("depth", C.c_void_p), ("conic_opacity", C.c_void_p),
                ("rgb", C.c_void_p), ("radius", C.c_void_p), ("tiles_touched", C.c_void_p),
                ("clamp", C.c_void_p), ("blend", C.c_void_p)]


class BinningS(C.Structure):
    _fields_ = [("keys", C.c_void_p), ("vals", C.c_void_p), ("tile_ranges", C.c_void_p),
                ("capacity", C.c_uint64), ("num_intersections", C.c_void_p), ("slot_order", C.c_void_p)]


class PartialS(C.Structure):
    _fields_ = [("ct", C.c_void_p), ("d", C.c_void_p), ("n_contrib", C.c_void_p)]


class PlanS(C.Structure):
    _fields_ = [("n_views", C.c_int32), ("cams", C.c_void_p), ("view_of_part", C.c_void_p),
                ("tile_state", C.c_void_p), ("flags", C.c_int32), ("max_scale", C.c_void_p), ("open_slots", C.c_int32),
                ("slot_map", C.c_void_p)]


class FrontsetS(C.Structure):
    _fields_ = [("proj", ProjectedS), ("bins", BinningS), ("ws", C.c_void_p), ("ws_bytes", C.c_size_t)]


class TrainsetS(C.Structure):
    _fields_ = [("params", GaussiansS), ("grads", GaussiansS), ("K", C.c_int32), ("part_offsets", C.c_void_p),
                ("sh_degree", C.c_int32), ("bg", C.c_float * 3), ("front", FrontsetS * 2), ("partials", PartialS),
                ("g_ct", C.c_void_p), ("g2d", C.c_void_p), ("images", C.c_void_p), ("T_totals", C.c_void_p),
                ("targets", C.c_void_p), ("g_images", C.c_void_p), ("dssim_ws", C.c_void_p), ("loss_sum", C.c_void_p),
                ("max_views", C.c_int32), ("cross_mask", C.c_void_p), ("touched", C.c_void_p)]


class BucketS(C.Structure):
    _fields_ = [("plan", PlanS), ("view_index", C.c_void_p), ("tile_state_out", C.c_void_p),
                ("part_depth_range", C.c_void_p)]


class AdamCfgS(C.Structure):
    _fields_ = [("param", C.c_void_p), ("grad", C.c_void_p), ("m", C.c_void_p), ("v", C.c_void_p),
                ("n_groups", C.c_int32), ("group_offsets", C.c_void_p), ("lr", C.c_void_p),
                ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float), ("step", C.c_int32),
                ("widths", C.c_void_p), ("sparse", C.c_int32), ("m_soa", GaussiansS), ("v_soa", GaussiansS)]


class IterOptsS(C.Structure):
    _fields_ = [("flags", C.c_int32), ("sat_eps", C.c_float), ("lambda_dssim", C.c_float)]


ITER_HOST = 1
ITER_FUSED_PROJECTION = 4
ITER_KEEP_ZERO_ROWS = 8


def lib():
    """Load libsplx.so; raise loudly if it is missing (the product path has no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: build it with "
                              "`python -m paper_2606_18588_b200.build` (nvcc, sm_100a). No CPU fallback exists.")
        L = C.CDLL(LIB_PATH)
        L.splx_last_error.restype = C.c_char_p
        L.splx_last_error.argtypes = [C.c_void_p]
        L.splx_launch_count.restype = C.c_int64
        L.splx_launch_count.argtypes = [C.c_void_p]
        L.splx_slot_map_words.restype = C.c_size_t
        L.splx_slot_map_words.argtypes = [C.c_int, C.c_void_p]
        L.splx_slot_map.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.splx_bin_sort_ws_bytes.restype = C.c_size_t
        L.splx_bin_sort_ws_bytes.argtypes = [C.c_int64, C.c_uint64, C.c_int, C.c_void_p]
        L.splx_backward_ws_bytes.restype = C.c_size_t
        L.splx_backward_ws_bytes.argtypes = [C.c_int64, C.c_int, C.c_void_p]
        L.splx_create.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.splx_destroy.argtypes = [C.c_void_p]
        L.splx_set_stream.argtypes = [C.c_void_p, C.c_void_p]
        L.splx_project.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.splx_bin_sort.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int, C.c_void_p, C.c_void_p,
                                    C.c_void_p, C.c_void_p, C.c_size_t]
        L.splx_check_capacity.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.splx_render_partial.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                          C.c_void_p, C.c_void_p]
        L.splx_compose.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                   C.c_void_p]
        L.splx_l1_loss_grad.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_float,
                                        C.c_void_p, C.c_void_p]
        L.splx_compose_backward.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                            C.c_void_p, C.c_void_p, C.c_void_p]
        L.splx_raster_backward.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                           C.c_void_p, C.c_void_p, C.c_void_p]
        L.splx_project_backward.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                            C.c_void_p, C.c_int, C.c_void_p]
        L.splx_backward.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                    C.c_void_p, C.c_size_t, C.c_int]
        L.splx_adam.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64,
                                C.c_float, C.c_float, C.c_float, C.c_float, C.c_int, C.c_float, C.c_int]
        L.splx_adam_groups.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int,
                                       C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_int,
                                       C.c_float, C.c_int]
        vp = C.c_void_p
        L.splx_visible_regions.argtypes = [C.c_int, C.c_int, vp, vp, vp, vp, vp, vp, vp, vp]
        L.splx_dssim_ws_floats.restype = C.c_size_t
        L.splx_dssim_ws_floats.argtypes = [vp]
        L.splx_dssim_loss_grad.argtypes = [vp, C.c_int, vp, vp, vp, C.c_float, C.c_float, vp, vp, vp]
        L.splx_dssim_loss_grad_static.argtypes = [vp, C.c_int, vp, vp, vp, C.c_float, C.c_float, vp, vp]
        L.splx_adam_groups_flagged.argtypes = [vp, vp, vp, vp, vp, C.c_int, vp, vp, C.c_int64, vp, vp, C.c_float, C.c_float,
                                               C.c_float, C.c_int, C.c_float]
        L.splx_microbench.argtypes = [vp, C.c_int, C.c_int64, vp, vp]
        L.splx_iteration.argtypes = [vp, vp, C.c_int, vp, C.c_int, vp, vp, vp, vp, vp, vp]
        L.splx_schedule_views.argtypes = [C.c_int, vp, C.c_int, vp, vp]
        L.splx_project_plan.argtypes = [vp, vp, C.c_int, vp, vp, C.c_int, vp]
        L.splx_bin_sort_plan.argtypes = [vp, vp, C.c_int64, C.c_int, vp, vp, vp, vp, C.c_size_t]
        L.splx_project_geometry_plan.argtypes = [vp, vp, C.c_int, vp, vp, vp]
        L.splx_project_colour_list_plan.argtypes = [vp, vp, C.c_int, vp, vp, C.c_int, vp, vp, vp]
        L.splx_render_partial_plan.argtypes = [vp, vp, vp, C.c_int, vp, vp, vp]
        L.splx_compose_plan.argtypes = [vp, C.c_int, vp, vp, vp, vp, vp, vp, C.c_float, vp]
        L.splx_compose_backward_plan.argtypes = [vp, C.c_int, vp, vp, vp, vp, vp, vp, vp]
        L.splx_compose_l1_backward_plan.argtypes = [vp, C.c_int, vp, vp, vp, vp, vp, C.c_float, vp, vp, vp, vp,
                                                    C.c_float, vp]
        L.splx_raster_backward_plan.argtypes = [vp, vp, vp, C.c_int, vp, vp, vp, vp]
        L.splx_project_backward_plan.argtypes = [vp, vp, C.c_int, vp, vp, C.c_int, vp, vp, C.c_int, vp]
        L.splx_backward_plan.argtypes = [vp, C.c_int, vp, vp, vp, vp, vp, vp, vp, vp, vp, C.c_int, vp, vp,
                                         C.c_size_t, C.c_int]
        L.splx_bin_sort_visible.argtypes = [vp, C.c_int64, C.c_uint64, C.c_int, vp, vp, vp]
        L.splx_bin_sort_gradient_rows.argtypes = [vp, vp, C.c_int64, C.c_uint64, C.c_int, vp, vp, vp, vp]
        L.splx_project_backward_list_plan.argtypes = [vp, vp, C.c_int, vp, vp, C.c_int, vp, vp, C.c_int, vp, vp, vp, vp]
        L.splx_adam_sparse.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.c_float, C.c_float, C.c_float, C.c_int, C.c_float]
        L.splx_cross_sets.argtypes = [vp, vp, C.c_int, vp, vp, vp, C.c_float, vp]
        L.splx_cross_depth_ranges.argtypes = [C.c_int, vp, vp, vp, vp]
        L.splx_bin_sort_filtered_plan.argtypes = [vp, vp, C.c_int64, C.c_int, vp, vp, vp, vp, vp, vp, C.c_size_t]
        _lib = L
    return _lib


def _ptr(t):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device tensors must be contiguous CUDA tensors"
    return t.data_ptr()


def camera_struct(cam) -> CameraS:
    """cam: any object with R, t, fx, fy, cx, cy, width, height, near_z (scenes.Camera)."""
    s = CameraS()
    R = [float(x) for x in list(cam.R.reshape(-1))]
    t = [float(x) for x in list(cam.t.reshape(-1))]
    s.R[:] = R
    s.t[:] = t
    s.fx, s.fy, s.cx, s.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    s.width, s.height, s.near_z = int(cam.width), int(cam.height), float(cam.near_z)
    return s


class Plan:
    """splx_plan: B views of one size, the view each partition renders (-1 = not a participant), the
    optional device tile-state bytes [K*tiles] and the flags.  Keeps the ctypes storage alive."""

    def __init__(self, cams, view_of_part, tile_state=None, sparse=False, max_scale=None, open_slots=0, slot_map=None):
        self.cams = list(cams)
        self.view_of_part = [int(v) for v in view_of_part]
        self.tile_state = tile_state
        self.flags = PLAN_SPARSE if sparse else 0
        self._cams = (CameraS * len(self.cams))(*[camera_struct(c) for c in self.cams])
        self._vop = (C.c_int32 * len(self.view_of_part))(*self.view_of_part)
        self._ms = None if max_scale is None else (C.c_float * len(self.view_of_part))(*[float(x) for x in max_scale])
        self._s = PlanS(len(self.cams), C.cast(self._cams, C.c_void_p), C.cast(self._vop, C.c_void_p),
                        _ptr(tile_state), self.flags, C.cast(self._ms, C.c_void_p) if self._ms is not None else None,
                        int(open_slots), _ptr(slot_map))
        self.open_slots = int(open_slots)
        self.slot_map = slot_map

    @property
    def K(self):
        return len(self.view_of_part)

    @property
    def B(self):
        return len(self.cams)

    def ref(self):
        return C.byref(self._s)


def visible_regions(aabb_lo, aabb_hi, cam, max_scale=None, box_part=None, K=None, cfg=None):
    """splx_visible_regions (host computation): returns (tile_state uint8 numpy [K, tiles], participants bitmask).
    max_scale: float[n_boxes] largest scale of the Gaussians with their mean in box j -> the conservative regions of
    reading s21 (None: the plain projected boxes); box_part: int[n_boxes] partition of every box (None: one box per
    partition); K: number of partitions; cfg: the splx_config tuple (None = defaults)."""
    import numpy as np
    lo = np.ascontiguousarray(aabb_lo, np.float32).reshape(-1, 3)
    hi = np.ascontiguousarray(aabb_hi, np.float32).reshape(-1, 3)
    nb = lo.shape[0]
    bp = np.ascontiguousarray(box_part, np.int32).reshape(nb) if box_part is not None else None
    if K is None:
        K = nb if bp is None else int(bp.max()) + 1
    TX, TY = (int(cam.width) + TILE - 1) // TILE, (int(cam.height) + TILE - 1) // TILE
    out = np.empty((K, TX * TY), np.uint8)
    part = C.c_uint64(0)
    cs = camera_struct(cam)
    ms = np.ascontiguousarray(max_scale, np.float32).reshape(nb) if max_scale is not None else None
    c = Config(*cfg) if cfg is not None else None
    rc = lib().splx_visible_regions(K, nb, bp.ctypes.data if bp is not None else None, lo.ctypes.data, hi.ctypes.data,
                                    ms.ctypes.data if ms is not None else None, C.byref(c) if c is not None else None,
                                    C.byref(cs), out.ctypes.data, C.byref(part))
    if rc != OK:
        raise SplxError(rc, "splx_visible_regions: invalid argument")
    return out, int(part.value)


def cross_depth_ranges(aabb_lo, aabb_hi, plan):
    """splx_cross_depth_ranges (host computation): D^k of every partition under the view it renders, float32 [K, 2]."""
    import numpy as np
    lo = np.ascontiguousarray(aabb_lo, np.float32).reshape(-1, 3)
    hi = np.ascontiguousarray(aabb_hi, np.float32).reshape(-1, 3)
    out = np.empty((lo.shape[0], 2), np.float32)
    rc = lib().splx_cross_depth_ranges(lo.shape[0], lo.ctypes.data, hi.ctypes.data, plan.ref(), out.ctypes.data)
    if rc != OK:
        raise SplxError(rc, "splx_cross_depth_ranges: invalid argument")
    return out


def schedule_views(participants, max_views_per_bucket=MAX_VIEWS):
    """splx_schedule_views (host computation): greedy conflict-free bucketing; returns bucket index per view."""
    n = len(participants)
    pa = (C.c_uint64 * max(n, 1))(*[int(x) for x in participants])
    out = (C.c_int32 * max(n, 1))()
    nb = C.c_int32(0)
    rc = lib().splx_schedule_views(n, pa, int(max_views_per_bucket), out, C.byref(nb))
    if rc != OK:
        raise SplxError(rc, "splx_schedule_views: invalid argument")
    return [int(out[i]) for i in range(n)], int(nb.value)


def gaussians_struct(p: dict, cls=GaussiansS):
    n = p["opacity_logit"].numel()
    for k, w in (("mean", 3), ("log_scale", 3), ("quat", 4), ("opacity_logit", 1), ("sh", 48)):
        assert p[k].dtype == torch.float32 and p[k].numel() == n * w, k
    return cls(_ptr(p["mean"]), _ptr(p["log_scale"]), _ptr(p["quat"]), _ptr(p["opacity_logit"]),
               _ptr(p["sh"]), n)


class Projected:
    def __init__(self, n, device):
        f = dict(dtype=torch.float32, device=device)
        self.n = n
        n = max(n, 1)            # keep every pointer non-null for an empty scene
        self.means2d = torch.empty((n, 2), **f)
        self.depth = torch.empty(n, **f)
        self.conic_opacity = torch.empty((n, 4), **f)
        self.rgb = torch.empty((n, 3), **f)
        self.radius = torch.empty(n, dtype=torch.int32, device=device)
        self.tiles_touched = torch.empty(n, dtype=torch.int32, device=device)  # uint32 bits
        self.clamp = torch.empty(n, dtype=torch.uint8, device=device)
        self.blend = torch.empty((n, BLEND_STRIDE), **f)

    def struct(self):
        return ProjectedS(_ptr(self.means2d), _ptr(self.depth), _ptr(self.conic_opacity), _ptr(self.rgb),
                          _ptr(self.radius), _ptr(self.tiles_touched), _ptr(self.clamp), _ptr(self.blend))


class Binning:
    def __init__(self, capacity, K, width, height, device):
        self.TX, self.TY = (width + TILE - 1) // TILE, (height + TILE - 1) // TILE
        self.capacity = int(capacity)
        self.keys = torch.empty(max(self.capacity, 2), dtype=torch.int64, device=device)     # uint64 bits
        self.vals = torch.empty(max(self.capacity, 4), dtype=torch.int32, device=device)     # uint32 bits
        self.tile_ranges = torch.zeros((K * self.TX * self.TY, 2), dtype=torch.int32, device=device)
        self.num_intersections = torch.zeros(2, dtype=torch.int64, device=device)
        #: slots by descending list length (splx_binning.slot_order); set to None to hand out CTAs in tile order
        self.slot_order = torch.zeros(K * self.TX * self.TY + ORDER_EXTRA, dtype=torch.int32, device=device)

    def struct(self):
        return BinningS(_ptr(self.keys), _ptr(self.vals), _ptr(self.tile_ranges), self.capacity,
                        _ptr(self.num_intersections), _ptr(self.slot_order))


class Partial:
    def __init__(self, K, width, height, device):
        self.ct = torch.empty((K, height, width, 4), dtype=torch.float32, device=device)
        self.d = torch.empty((K, height, width), dtype=torch.float32, device=device)
        self.n_contrib = torch.empty((K, height, width), dtype=torch.int32, device=device)

    def struct(self):
        return PartialS(_ptr(self.ct), _ptr(self.d), _ptr(self.n_contrib))


class Context:
    """One splx_ctx bound to a device and a CUDA stream (default: torch's current stream)."""

    def __init__(self, device=0, stream=None, cfg=None):
        L = lib()
        if not torch.cuda.is_available():
            raise SplxError(ERR_CUDA, "no CUDA device; libsplx has no CPU fallback")
        self.device = torch.device("cuda", device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device).cuda_stream
        self._h = C.c_void_p()
        c = Config(*cfg) if cfg is not None else None
        rc = L.splx_create(C.byref(self._h), device, C.c_void_p(stream), C.byref(c) if c is not None else None)
        if rc != OK:
            raise SplxError(rc, L.splx_last_error(None).decode())

    def close(self):
        if getattr(self, "_h", None):
            lib().splx_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != OK:
            raise SplxError(rc, lib().splx_last_error(self._h).decode())

    def set_stream(self, stream):
        self._check(lib().splx_set_stream(self._h, C.c_void_p(stream)))

    def launch_count(self) -> int:
        return int(lib().splx_launch_count(self._h))

    # ---- the calls of SURVEY.md s8(b) ---------------------------------------------------
    def project(self, params: dict, cam, sh_degree: int, out: Projected):
        g = gaussians_struct(params)
        cs = camera_struct(cam)
        ps = out.struct()
        self._check(lib().splx_project(self._h, C.byref(g), C.byref(cs), sh_degree, C.byref(ps)))

    def bin_sort_ws_bytes(self, n, capacity, K, cam) -> int:
        cs = camera_struct(cam)
        return int(lib().splx_bin_sort_ws_bytes(n, capacity, K, C.byref(cs)))

    def bin_sort(self, proj: Projected, K: int, part_offsets, cam, out: Binning, ws: torch.Tensor):
        offs = (C.c_int64 * (K + 1))(*[int(x) for x in part_offsets])
        cs = camera_struct(cam)
        ps, bs = proj.struct(), out.struct()
        self._check(lib().splx_bin_sort(self._h, C.byref(ps), proj.n, K, offs, C.byref(cs), C.byref(bs),
                                        _ptr(ws), ws.numel() * ws.element_size()))

    def check_capacity(self, bins: Binning) -> int:
        m = C.c_uint64(0)
        bs = bins.struct()
        self._check(lib().splx_check_capacity(self._h, C.byref(bs), C.byref(m)))
        return int(m.value)

    def render_partial(self, proj: Projected, bins: Binning, K: int, cam, out: Partial, pairs=None):
        cs = camera_struct(cam)
        ps, bs, os_ = proj.struct(), bins.struct(), out.struct()
        self._check(lib().splx_render_partial(self._h, C.byref(ps), C.byref(bs), K, C.byref(cs), C.byref(os_),
                                              _ptr(pairs)))

    def compose(self, K: int, partials: Partial, cam, bg, image: torch.Tensor, T_total=None):
        cs = camera_struct(cam)
        b = (C.c_float * 3)(*[float(x) for x in bg])
        ps = partials.struct()
        self._check(lib().splx_compose(self._h, K, C.byref(ps), C.byref(cs), b, _ptr(image), _ptr(T_total)))

    def l1_loss_grad(self, image, target, g_image, loss_sum=None, scale=1.0):
        self._check(lib().splx_l1_loss_grad(self._h, _ptr(image), _ptr(target), image.numel(), scale,
                                            _ptr(g_image), _ptr(loss_sum)))

    def compose_backward(self, K, partials: Partial, cam, bg, g_image, g_T_total, g_ct):
        cs = camera_struct(cam)
        b = (C.c_float * 3)(*[float(x) for x in bg])
        ps = partials.struct()
        self._check(lib().splx_compose_backward(self._h, K, C.byref(ps), C.byref(cs), b, _ptr(g_image),
                                                _ptr(g_T_total), _ptr(g_ct)))

    def raster_backward(self, proj: Projected, bins: Binning, K, cam, partials: Partial, g_ct, g2d):
        cs = camera_struct(cam)
        ps, bs, pa = proj.struct(), bins.struct(), partials.struct()
        self._check(lib().splx_raster_backward(self._h, C.byref(ps), C.byref(bs), K, C.byref(cs), C.byref(pa),
                                               _ptr(g_ct), _ptr(g2d)))

    def project_backward(self, params: dict, cam, sh_degree, proj: Projected, g2d, grads: dict, clear_g2d=False,
                         overwrite=False):
        g = gaussians_struct(params)
        gg = gaussians_struct(grads)
        cs = camera_struct(cam)
        ps = proj.struct()
        self._check(lib().splx_project_backward(self._h, C.byref(g), C.byref(cs), sh_degree, C.byref(ps),
                                                _ptr(g2d), (PB_CLEAR_G2D if clear_g2d else 0) | (PB_OVERWRITE if overwrite else 0),
                                                C.byref(gg)))

    def backward_ws_bytes(self, n, K, cam) -> int:
        cs = camera_struct(cam)
        return int(lib().splx_backward_ws_bytes(n, K, C.byref(cs)))

    def backward(self, K, partials: Partial, cam, bg, g_image, g_T_total, params: dict, proj: Projected,
                 bins: Binning, sh_degree, grads: dict, ws: torch.Tensor, overwrite=False):
        cs = camera_struct(cam)
        b = (C.c_float * 3)(*[float(x) for x in bg])
        pa, ps, bs = partials.struct(), proj.struct(), bins.struct()
        g, gg = gaussians_struct(params), gaussians_struct(grads)
        self._check(lib().splx_backward(self._h, K, C.byref(pa), C.byref(cs), b, _ptr(g_image), _ptr(g_T_total),
                                        C.byref(g), C.byref(ps), C.byref(bs), sh_degree, C.byref(gg),
                                        _ptr(ws), ws.numel() * ws.element_size(), PB_OVERWRITE if overwrite else 0))

    def adam(self, param, grad, m, v, lr, beta1=0.9, beta2=0.999, eps=1e-15, step=1, grad_scale=1.0,
             zero_grad=False):
        self._check(lib().splx_adam(self._h, _ptr(param), _ptr(grad), _ptr(m), _ptr(v), param.numel(), lr,
                                    beta1, beta2, eps, step, grad_scale, int(zero_grad)))

    def adam_groups(self, param, grad, m, v, group_offsets, lrs, beta1=0.9, beta2=0.999, eps=1e-15, step=1,
                    grad_scale=1.0, zero_grad=False):
        n = len(lrs)
        offs = (C.c_int64 * (n + 1))(*[int(x) for x in group_offsets])
        lr = (C.c_float * n)(*[float(x) for x in lrs])
        self._check(lib().splx_adam_groups(self._h, _ptr(param), _ptr(grad), _ptr(m), _ptr(v), n, offs, lr,
                                           beta1, beta2, eps, step, grad_scale, int(zero_grad)))

    def adam_groups_flagged(self, param, grad, m, v, group_offsets, widths, rows, touched, lrs, beta1=0.9, beta2=0.999,
                            eps=1e-15, step=1, grad_scale=1.0):
        n = len(lrs)
        offs = (C.c_int64 * (n + 1))(*[int(x) for x in group_offsets])
        wd = (C.c_int32 * n)(*[int(x) for x in widths])
        lr = (C.c_float * n)(*[float(x) for x in lrs])
        self._check(lib().splx_adam_groups_flagged(self._h, _ptr(param), _ptr(grad), _ptr(m), _ptr(v), n, offs, wd, int(rows),
                                                   _ptr(touched), lr, beta1, beta2, eps, step, grad_scale))

    @staticmethod
    def slot_map_words(K, cam) -> int:
        cs = camera_struct(cam)
        return int(lib().splx_slot_map_words(int(K), C.byref(cs)))

    def slot_map(self, plan: "Plan", device=None):
        """splx_slot_map: the numbering of the plan's open slots (a new device tensor), for Plan(..., slot_map=...)."""
        words = self.slot_map_words(plan.K, plan.cams[0])
        out = torch.empty(words, dtype=torch.int32, device=plan.tile_state.device if device is None else device)
        self._check(lib().splx_slot_map(self._h, plan.K, plan.ref(), _ptr(out)))
        return out

    # ---- the same stages under a launch plan (visibility prediction, consolidated views) ---------
    visible_regions = staticmethod(visible_regions)     # host computations: no context needed
    schedule_views = staticmethod(schedule_views)

    @staticmethod
    def _offs(part_offsets):
        return (C.c_int64 * len(part_offsets))(*[int(x) for x in part_offsets])

    def project_plan(self, params: dict, part_offsets, plan: Plan, sh_degree: int, out: Projected):
        g, ps = gaussians_struct(params), out.struct()
        self._check(lib().splx_project_plan(self._h, C.byref(g), plan.K, self._offs(part_offsets), plan.ref(),
                                            sh_degree, C.byref(ps)))

    def project_geometry_plan(self, params: dict, part_offsets, plan: Plan, out: Projected):
        g, ps = gaussians_struct(params), out.struct()
        self._check(lib().splx_project_geometry_plan(self._h, C.byref(g), plan.K, self._offs(part_offsets), plan.ref(), C.byref(ps)))

    def project_colour_list_plan(self, params: dict, part_offsets, plan: Plan, sh_degree: int, out: Projected,
                                 visible_ptr: int, count_ptr: int):
        g, ps = gaussians_struct(params), out.struct()
        self._check(lib().splx_project_colour_list_plan(self._h, C.byref(g), plan.K, self._offs(part_offsets), plan.ref(), sh_degree,
                                                        C.byref(ps), C.c_void_p(visible_ptr), C.c_void_p(count_ptr)))

    def bin_sort_plan(self, proj: Projected, part_offsets, plan: Plan, out: Binning, ws: torch.Tensor):
        ps, bs = proj.struct(), out.struct()
        self._check(lib().splx_bin_sort_plan(self._h, C.byref(ps), proj.n, plan.K, self._offs(part_offsets), plan.ref(),
                                             C.byref(bs), _ptr(ws), ws.numel() * ws.element_size()))

    def cross_sets(self, params: dict, part_offsets, cell_lo, cell_hi, cross_mask: torch.Tensor, support_sigma=3.0):
        """splx_cross_sets: cross_mask = device int64/uint64 [n] (bit s = in Q_cross against partition s)."""
        import numpy as np
        lo = np.ascontiguousarray(cell_lo, np.float32).reshape(-1, 3)
        hi = np.ascontiguousarray(cell_hi, np.float32).reshape(-1, 3)
        g = gaussians_struct(params)
        self._check(lib().splx_cross_sets(self._h, C.byref(g), lo.shape[0], self._offs(part_offsets), lo.ctypes.data,
                                          hi.ctypes.data, float(support_sigma), _ptr(cross_mask)))

    def bin_sort_filtered_plan(self, proj: Projected, part_offsets, plan: Plan, cross_mask, part_depth_range, out: Binning,
                               ws: torch.Tensor):
        import numpy as np
        ps, bs = proj.struct(), out.struct()
        zr = np.ascontiguousarray(part_depth_range, np.float32).reshape(-1)
        self._check(lib().splx_bin_sort_filtered_plan(self._h, C.byref(ps), proj.n, plan.K, self._offs(part_offsets),
                                                      plan.ref(), _ptr(cross_mask), zr.ctypes.data, C.byref(bs), _ptr(ws),
                                                      ws.numel() * ws.element_size()))

    cross_depth_ranges = staticmethod(cross_depth_ranges)

    def render_partial_plan(self, proj: Projected, bins: Binning, plan: Plan, out: Partial, pairs=None):
        ps, bs, os_ = proj.struct(), bins.struct(), out.struct()
        self._check(lib().splx_render_partial_plan(self._h, C.byref(ps), C.byref(bs), plan.K, plan.ref(), C.byref(os_),
                                                   _ptr(pairs)))

    def compose_plan(self, partials: Partial, bins, plan: Plan, bg, image, T_total=None, sat_eps=1e-4,
                     tile_state_out=None):
        b = (C.c_float * 3)(*[float(x) for x in bg])
        ps = partials.struct()
        bs = bins.struct() if bins is not None else None
        self._check(lib().splx_compose_plan(self._h, plan.K, C.byref(ps), C.byref(bs) if bs is not None else None,
                                            plan.ref(), b, _ptr(image), _ptr(T_total), float(sat_eps),
                                            _ptr(tile_state_out)))

    def compose_l1_backward_plan(self, partials: Partial, bins, plan: Plan, bg, targets, image, T_total, loss_sum, g_ct,
                                 scale=1.0, sat_eps=1e-4, tile_state_out=None):
        b = (C.c_float * 3)(*[float(x) for x in bg])
        ps = partials.struct()
        bs = bins.struct() if bins is not None else None
        self._check(lib().splx_compose_l1_backward_plan(self._h, plan.K, C.byref(ps), C.byref(bs) if bs is not None else None,
                                                        plan.ref(), b, _ptr(targets), float(scale), _ptr(image),
                                                        _ptr(T_total), _ptr(loss_sum), _ptr(g_ct), float(sat_eps),
                                                        _ptr(tile_state_out)))

    def compose_backward_plan(self, partials: Partial, bins, plan: Plan, bg, g_image, g_T_total, g_ct):
        b = (C.c_float * 3)(*[float(x) for x in bg])
        ps = partials.struct()
        bs = bins.struct() if bins is not None else None
        self._check(lib().splx_compose_backward_plan(self._h, plan.K, C.byref(ps), C.byref(bs) if bs is not None else None,
                                                     plan.ref(), b, _ptr(g_image), _ptr(g_T_total), _ptr(g_ct)))

    def raster_backward_plan(self, proj: Projected, bins: Binning, plan: Plan, partials: Partial, g_ct, g2d):
        ps, bs, pa = proj.struct(), bins.struct(), partials.struct()
        self._check(lib().splx_raster_backward_plan(self._h, C.byref(ps), C.byref(bs), plan.K, plan.ref(), C.byref(pa),
                                                    _ptr(g_ct), _ptr(g2d)))

    def project_backward_plan(self, params: dict, part_offsets, plan: Plan, sh_degree, proj: Projected, g2d,
                              grads: dict, clear_g2d=False, overwrite=False):
        g, gg, ps = gaussians_struct(params), gaussians_struct(grads), proj.struct()
        flags = (PB_CLEAR_G2D if clear_g2d else 0) | (PB_OVERWRITE if overwrite else 0)
        self._check(lib().splx_project_backward_plan(self._h, C.byref(g), plan.K, self._offs(part_offsets), plan.ref(),
                                                     sh_degree, C.byref(ps), _ptr(g2d), flags, C.byref(gg)))

    @staticmethod
    def bin_sort_visible(ws: torch.Tensor, n, capacity, K, cam):
        """Device pointers (ints) of the visible list and of its count inside the bin_sort workspace."""
        cs = camera_struct(cam)
        lst, cnt = C.c_void_p(), C.c_void_p()
        rc = lib().splx_bin_sort_visible(_ptr(ws), n, capacity, K, C.byref(cs), C.byref(lst), C.byref(cnt))
        if rc != OK:
            raise SplxError(rc, "splx_bin_sort_visible: invalid argument")
        return lst.value, cnt.value

    def bin_sort_gradient_rows(self, ws: torch.Tensor, n, capacity, K, cam, g2d):
        """splx_bin_sort_gradient_rows: device pointers (ints) of the list of Gaussians with a non-zero g2d row and of its count."""
        cs = camera_struct(cam)
        lst, cnt = C.c_void_p(), C.c_void_p()
        self._check(lib().splx_bin_sort_gradient_rows(self._h, _ptr(ws), n, capacity, K, C.byref(cs), _ptr(g2d), C.byref(lst), C.byref(cnt)))
        return lst.value, cnt.value

    def project_backward_list_plan(self, params: dict, part_offsets, plan: Plan, sh_degree, proj: Projected, g2d,
                                   grads: dict, visible_ptr: int, count_ptr: int, clear_g2d=False, touched=None):
        g, gg, ps = gaussians_struct(params), gaussians_struct(grads), proj.struct()
        self._check(lib().splx_project_backward_list_plan(self._h, C.byref(g), plan.K, self._offs(part_offsets), plan.ref(),
                                                          sh_degree, C.byref(ps), _ptr(g2d), PB_CLEAR_G2D if clear_g2d else 0,
                                                          C.byref(gg), C.c_void_p(visible_ptr), C.c_void_p(count_ptr),
                                                          _ptr(touched)))

    def adam_sparse(self, params: dict, grads: dict, m: dict, v: dict, touched, lrs, beta1=0.9, beta2=0.999, eps=1e-15,
                    step=1, grad_scale=1.0):
        sets = [gaussians_struct(x) for x in (params, grads, m, v)]
        lr = (C.c_float * 5)(*[float(x) for x in lrs])
        self._check(lib().splx_adam_sparse(self._h, C.byref(sets[0]), C.byref(sets[1]), C.byref(sets[2]), C.byref(sets[3]),
                                           _ptr(touched), lr, beta1, beta2, eps, int(step), float(grad_scale)))

    @staticmethod
    def dssim_ws_floats(width, height) -> int:
        cs = CameraS()
        cs.width, cs.height = int(width), int(height)
        return int(lib().splx_dssim_ws_floats(C.byref(cs)))

    def dssim_loss_grad(self, cam, image, target, g_image, loss_sum, ws, lam, scale=None):
        """splx_dssim_loss_grad: image / target / g_image [B,H,W,3] (or [H,W,3]); loss_sum device double[2] or None."""
        B = image.shape[0] if image.dim() == 4 else 1
        cs = camera_struct(cam)
        self._check(lib().splx_dssim_loss_grad(self._h, B, C.byref(cs), _ptr(image), _ptr(target), float(lam),
                                               float(B if scale is None else scale), _ptr(g_image), _ptr(loss_sum), _ptr(ws)))

    def dssim_loss_grad_static(self, cam, image, target, g_image, loss_sum, lam, scale=None):
        """splx_dssim_loss_grad_static: the same with the scratch in the library's static device array (no allocation;
        n_views * W * H <= DSSIM_STATIC_MAX_PIXELS)."""
        B = image.shape[0] if image.dim() == 4 else 1
        cs = camera_struct(cam)
        self._check(lib().splx_dssim_loss_grad_static(self._h, B, C.byref(cs), _ptr(image), _ptr(target), float(lam),
                                                      float(B if scale is None else scale), _ptr(g_image), _ptr(loss_sum)))

    def iteration(self, trainset: "TrainsetS", buckets, n_views, targets, images_out=None, loss_out=None, m_out=None,
                  host=False, sat_eps=1e-4, lambda_dssim=0.0, adam: "AdamCfgS" = None, fused_projection=False, keep_zero_rows=False):
        """splx_iteration.  buckets: ctypes array of BucketS; targets / images_out: lists of raw pointers (ints; device
        pointers, or pinned host pointers with host=True); loss_out / m_out: raw pinned host pointers or None."""
        tg = (C.c_void_p * n_views)(*[C.c_void_p(int(x)) for x in targets])
        io = None
        if images_out is not None:
            io = (C.c_void_p * n_views)(*[C.c_void_p(int(x)) if x else None for x in images_out])
        opts = IterOptsS((ITER_HOST if host else 0) | (ITER_FUSED_PROJECTION if fused_projection else 0) |
                         (ITER_KEEP_ZERO_ROWS if keep_zero_rows else 0), float(sat_eps),
                         float(lambda_dssim))
        self._check(lib().splx_iteration(self._h, C.byref(trainset), len(buckets), buckets, int(n_views), tg, io,
                                         C.c_void_p(loss_out) if loss_out else None, C.c_void_p(m_out) if m_out else None,
                                         C.byref(opts), C.byref(adam) if adam is not None else None))

    def microbench(self, kind: int, iters: int, sink) -> float:
        """splx_microbench: launches the FMA (kind 0) or ex2 (kind 1) loop; returns the work of the launch (flops / ex2)."""
        w = C.c_double(0.0)
        self._check(lib().splx_microbench(self._h, int(kind), int(iters), _ptr(sink), C.byref(w)))
        return float(w.value)

    def backward_plan(self, part_offsets, plan: Plan, partials: Partial, bg, g_image, g_T_total, params: dict,
                      proj: Projected, bins: Binning, sh_degree, grads: dict, ws: torch.Tensor, overwrite=False):
        b = (C.c_float * 3)(*[float(x) for x in bg])
        pa, ps, bs = partials.struct(), proj.struct(), bins.struct()
        g, gg = gaussians_struct(params), gaussians_struct(grads)
        self._check(lib().splx_backward_plan(self._h, plan.K, self._offs(part_offsets), plan.ref(), C.byref(pa), b,
                                             _ptr(g_image), _ptr(g_T_total), C.byref(g), C.byref(ps), C.byref(bs),
                                             sh_degree, C.byref(gg), _ptr(ws), ws.numel() * ws.element_size(),
                                             PB_OVERWRITE if overwrite else 0))
