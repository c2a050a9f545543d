"""Thin Python binding of libnd_moc.so (include/nd.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for device memory
(the workspace and the phi/Q tensors) and the stream.  There is no CPU fallback: importing works on a CPU
box (the library loads and exports its symbols), but every compute call returns ND_ERR_CUDA without a B200.

Functions keep the C names: nd_tracks_generate, nd_problem_create, nd_transport_sweep, nd_source_update,
nd_power_iteration, ...  Cites: include/nd.h (which cites PAPER.md Eq. (1),(3)-(5), section III.A).
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libnd_moc.so")

ND_OK = 0
ND_ERR_WORKSPACE = 4
ND_ERR_NOT_CONVERGED = 7
ND_BC_VACUUM, ND_BC_REFLECTIVE = 0, 1
ND_EXP_FAST, ND_EXP_EXPM1 = 0, 1
ND_SWEEP_AUTO, ND_SWEEP_ATOMIC, ND_SWEEP_SWATH = 0, 1, 3

EXPORTS = [
    "nd_tracks_generate", "nd_tracks_device_workspace_bytes", "nd_tracks_generate_device", "nd_tracks_generate_resident", "nd_tracks_materialise", "nd_tracks_view", "nd_tracks_shard", "nd_tracks_destroy", "nd_tally_reducer_set", "nd_workspace_bytes", "nd_problem_create", "nd_problem_stream_view",
    "nd_problem_destroy", "nd_transport_sweep", "nd_source_update", "nd_power_iteration", "nd_state_reset",
    "nd_boundary_flux_fill", "nd_boundary_flux_get", "nd_boundary_flux_set", "nd_outgoing_flux_get", "nd_flux_get", "nd_flux_set",
    "nd_track_volume_get", "nd_tally_get", "nd_cmfd_surfaces", "nd_microbench", "nd_cmfd_workspace_bytes", "nd_cmfd_create",
    "nd_cmfd_destroy", "nd_cmfd_iteration", "nd_cmfd_sweep", "nd_cmfd_currents_get", "nd_cmfd_collapse", "nd_cmfd_coarse_get",
    "nd_cmfd_coarse_set", "nd_cmfd_solve", "nd_cmfd_prolong", "nd_p1_workspace_bytes", "nd_p1_create", "nd_p1_destroy",
    "nd_p1_transport_sweep", "nd_p1_source_update", "nd_p1_state_reset", "nd_p1_power_iteration", "nd_profile_enable", "nd_profile_read", "nd_sweep_phases_get", "nd_problem_info_get", "nd_fission_rate_static",
    "nd_swath_stream_build", "nd_swath_stream_view", "nd_swath_stream_destroy",
    "nd_status_string", "nd_last_error", "nd_version", "nd_build_id",
]


class NdError(RuntimeError):
    def __init__(self, status, where, message):
        super().__init__(f"{where}: {status} {message}")
        self.status = status


class nd_options(C.Structure):
    _fields_ = [("exp_mode", C.c_int32), ("sweep_kernel", C.c_int32),
                ("window_regions", C.c_int32), ("block_warps", C.c_int32), ("tile_segments", C.c_int32),
                ("delta_buffers", C.c_int32), ("blocks_per_sm", C.c_int32), ("tile_lag", C.c_int32), ("q_copies", C.c_int32), ("graph_mode", C.c_int32), ("cmfd_stream", C.c_int32), ("item_order", C.c_int32), ("p1_stream", C.c_int32), ("reserved", C.c_int32 * 3)]


class nd_mesh_desc(C.Structure):
    _fields_ = [("n_vertices", C.c_int32), ("n_triangles", C.c_int32), ("xy", C.c_void_p), ("tri", C.c_void_p),
                ("W", C.c_double), ("H", C.c_double), ("bc", C.c_int32 * 4)]


class nd_tracks_view_t(C.Structure):
    _fields_ = [("n_tracks", C.c_int32), ("n_regions", C.c_int32), ("n_segments", C.c_int64), ("n_half", C.c_int32),
                ("track_seg_offset", C.c_void_p), ("seg_region", C.c_void_p), ("seg_length", C.c_void_p),
                ("track_weight", C.c_void_p), ("link", C.c_void_p), ("track_azim", C.c_void_p),
                ("track_ends", C.c_void_p), ("track_volume", C.c_void_p), ("azim_phi", C.c_void_p),
                ("azim_weight", C.c_void_p), ("azim_spacing", C.c_void_p), ("track_global", C.c_void_p),
                ("seg_region_device", C.c_void_p), ("seg_length_device", C.c_void_p)]


class nd_stream_device_view_t(C.Structure):
    _fields_ = [("blob", C.c_void_p), ("blob_bytes", C.c_size_t), ("tile_ref", C.c_void_p), ("swath_tile0", C.c_void_p),
                ("swath_track", C.c_void_p), ("items", C.c_void_p), ("n_tiles", C.c_int64), ("n_swaths", C.c_int64),
                ("n_items", C.c_int64), ("tracks_per_swath", C.c_int32), ("built_on_device", C.c_int32)]


class nd_problem_desc(C.Structure):
    _fields_ = [("n_regions", C.c_int32), ("n_materials", C.c_int32), ("n_groups", C.c_int32), ("n_polar", C.c_int32),
                ("n_tracks", C.c_int32), ("region_material", C.c_void_p), ("sigma_t", C.c_void_p),
                ("sigma_s", C.c_void_p), ("nu_sigma_f", C.c_void_p), ("chi", C.c_void_p), ("polar_sin", C.c_void_p),
                ("polar_weight", C.c_void_p), ("track_seg_offset", C.c_void_p), ("seg_region", C.c_void_p),
                ("seg_length", C.c_void_p), ("track_weight", C.c_void_p), ("link", C.c_void_p),
                ("track_azim", C.c_void_p), ("track_ends", C.c_void_p), ("region_volume", C.c_void_p),
                ("seg_on_device", C.c_int32), ("reserved", C.c_int32)]


ND_TALLY_REDUCE_FN = C.CFUNCTYPE(C.c_int32, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p)


class nd_iter_stats(C.Structure):
    _fields_ = [("k_eff", C.c_double), ("fission_rate", C.c_double), ("dk", C.c_double), ("dphi_max", C.c_double),
                ("leakage", C.c_double), ("balance_residual", C.c_double)]


class nd_profile(C.Structure):
    _fields_ = [("sweep_ms", C.c_double), ("sweep_launches", C.c_int64), ("kernels_launched", C.c_int64)]


class nd_problem_info(C.Structure):
    _fields_ = [("n_segments", C.c_int64), ("n_segments_padded", C.c_int64), ("updates_per_sweep", C.c_int64),
                ("algorithmic_bytes", C.c_int64), ("group_stride", C.c_int32), ("sweep_kernel", C.c_int32),
                ("n_batches", C.c_int32), ("reserved", C.c_int32), ("mean_regions_per_tile", C.c_double),
                ("mean_segments_per_tile", C.c_double), ("lockstep_efficiency", C.c_double), ("block_threads", C.c_int32),
                ("smem_bytes", C.c_int32), ("grid_blocks", C.c_int32), ("tracks_per_block", C.c_int32)]


class nd_cmfd_options(C.Structure):
    _fields_ = [("tol", C.c_double), ("max_outer", C.c_int32), ("inner_sweeps", C.c_int32), ("relax", C.c_double),
                ("rel_tol", C.c_double), ("reserved", C.c_int32 * 2)]


class nd_cmfd_stats(C.Structure):
    _fields_ = [("k_sweep", C.c_double), ("k_eff", C.c_double), ("coarse_iters", C.c_int32), ("coarse_ok", C.c_int32)]


class nd_microbench_result(C.Structure):
    _fields_ = [("mufu_ex2_per_clk_per_sm", C.c_double), ("mufu_ex2_per_s", C.c_double), ("sm_clock_mhz", C.c_double),
                ("red_f64_l2_per_s", C.c_double), ("red_f64_hbm_per_s", C.c_double), ("n_sm", C.c_int32), ("reserved", C.c_int32)]


class nd_trace_timing(C.Structure):
    _fields_ = [("prepare_s", C.c_double), ("count_kernel_ms", C.c_double), ("fill_kernel_ms", C.c_double),
                ("copy_s", C.c_double), ("finish_s", C.c_double), ("total_s", C.c_double), ("n_segments", C.c_int64),
                ("batches", C.c_int32), ("reserved", C.c_int32)]


class nd_swath_stream_view_t(C.Structure):
    _fields_ = [("n_swaths", C.c_int64), ("n_tiles", C.c_int64), ("blob_bytes", C.c_int64), ("n_items", C.c_int64),
                ("blob", C.c_void_p), ("tile_ref", C.c_void_p), ("swath_tile0", C.c_void_p), ("swath_track", C.c_void_p),
                ("items", C.c_void_p), ("mean_regions_per_tile", C.c_double), ("mean_segments_per_tile", C.c_double),
                ("lockstep_efficiency", C.c_double), ("max_head_bytes", C.c_int32), ("max_rec_bytes", C.c_int32)]


_lib = None


def lib():
    """Load libnd_moc.so (built in-tree by paper_2607_01591_b200._build).  Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_2607_01591_b200._build` "
                              "(there is no CPU or PyTorch fallback for the MOC hot path)")
        L = C.CDLL(_LIB_PATH)
        L.nd_status_string.restype = C.c_char_p
        L.nd_status_string.argtypes = [C.c_int]
        L.nd_last_error.restype = C.c_char_p
        L.nd_last_error.argtypes = [C.c_void_p]
        L.nd_version.restype = C.c_uint32
        L.nd_build_id.restype = C.c_char_p
        L.nd_tracks_generate.argtypes = [C.POINTER(nd_mesh_desc), C.c_int32, C.c_double, C.c_int32, C.POINTER(C.c_void_p)]
        L.nd_tracks_device_workspace_bytes.argtypes = [C.POINTER(nd_mesh_desc), C.c_int32, C.c_double, C.POINTER(C.c_size_t),
                                                       C.POINTER(C.c_size_t)]
        L.nd_tracks_generate_device.argtypes = [C.POINTER(nd_mesh_desc), C.c_int32, C.c_double, C.c_void_p, C.c_size_t,
                                                C.c_void_p, C.POINTER(nd_trace_timing), C.POINTER(C.c_void_p)]
        L.nd_tracks_generate_resident.argtypes = [C.POINTER(nd_mesh_desc), C.c_int32, C.c_double, C.c_void_p, C.c_size_t,
                                                  C.c_void_p, C.c_void_p, C.POINTER(C.c_size_t), C.POINTER(C.c_void_p)]
        L.nd_tracks_materialise.argtypes = [C.c_void_p, C.c_void_p]
        L.nd_tracks_view.argtypes = [C.c_void_p, C.POINTER(nd_tracks_view_t)]
        L.nd_tracks_destroy.argtypes = [C.c_void_p]
        L.nd_tracks_shard.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.POINTER(C.c_void_p)]
        L.nd_tally_reducer_set.argtypes = [C.c_void_p, ND_TALLY_REDUCE_FN, C.c_void_p]
        L.nd_fission_rate_static.argtypes = [C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.nd_problem_stream_view.argtypes = [C.c_void_p, C.POINTER(nd_stream_device_view_t)]
        L.nd_workspace_bytes.argtypes = [C.POINTER(nd_problem_desc), C.POINTER(nd_options), C.POINTER(C.c_size_t)]
        L.nd_problem_create.argtypes = [C.POINTER(nd_problem_desc), C.POINTER(nd_options), C.c_void_p, C.c_size_t,
                                        C.c_void_p, C.POINTER(C.c_void_p)]
        L.nd_problem_destroy.argtypes = [C.c_void_p]
        L.nd_transport_sweep.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.nd_source_update.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.nd_power_iteration.argtypes = [C.c_void_p, C.c_int32, C.c_double, C.c_double, C.POINTER(C.c_double),
                                         C.c_void_p, C.POINTER(C.c_int32), C.c_void_p, C.c_void_p]
        L.nd_state_reset.argtypes = [C.c_void_p, C.c_void_p]
        L.nd_boundary_flux_fill.argtypes = [C.c_void_p, C.c_float, C.c_void_p]
        L.nd_boundary_flux_get.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.nd_boundary_flux_set.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.nd_outgoing_flux_get.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.nd_flux_get.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.nd_flux_set.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        L.nd_track_volume_get.argtypes = [C.c_void_p, C.c_void_p]
        L.nd_tally_get.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.nd_cmfd_surfaces.argtypes = [C.POINTER(nd_problem_desc), C.c_int32, C.c_void_p, C.c_int32, C.POINTER(C.c_int32),
                                       C.c_void_p, C.c_void_p]
        L.nd_microbench.argtypes = [C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(nd_microbench_result)]
        L.nd_cmfd_workspace_bytes.argtypes = [C.c_void_p, C.POINTER(nd_problem_desc), C.c_int32, C.c_void_p, C.c_int32,
                                              C.POINTER(C.c_size_t)]
        L.nd_cmfd_create.argtypes = [C.c_void_p, C.POINTER(nd_problem_desc), C.c_int32, C.c_void_p, C.c_int32, C.c_void_p,
                                     C.c_void_p, C.c_void_p, C.POINTER(nd_cmfd_options), C.c_void_p, C.c_size_t, C.c_void_p,
                                     C.POINTER(C.c_void_p)]
        L.nd_cmfd_destroy.argtypes = [C.c_void_p]
        L.nd_cmfd_iteration.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_double), C.c_void_p, C.c_void_p]
        L.nd_cmfd_sweep.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.nd_cmfd_currents_get.argtypes = [C.c_void_p] * 5
        L.nd_cmfd_collapse.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.nd_cmfd_coarse_get.argtypes = [C.c_void_p] * 8
        L.nd_cmfd_coarse_set.argtypes = [C.c_void_p] * 10
        L.nd_cmfd_solve.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double), C.c_void_p, C.POINTER(C.c_int32), C.c_void_p]
        L.nd_cmfd_prolong.argtypes = [C.c_void_p, C.c_void_p]
        L.nd_p1_workspace_bytes.argtypes = [C.c_void_p, C.POINTER(C.c_size_t)]
        L.nd_p1_create.argtypes = [C.c_void_p, C.POINTER(nd_problem_desc), C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p,
                                   C.POINTER(C.c_void_p)]
        L.nd_p1_destroy.argtypes = [C.c_void_p]
        L.nd_p1_transport_sweep.argtypes = [C.c_void_p] * 8
        L.nd_p1_source_update.argtypes = [C.c_void_p] * 4 + [C.c_double] + [C.c_void_p] * 4
        L.nd_p1_state_reset.argtypes = [C.c_void_p, C.c_void_p]
        L.nd_p1_power_iteration.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_double), C.c_void_p, C.c_void_p, C.c_void_p,
                                            C.c_void_p, C.c_void_p]
        L.nd_profile_enable.argtypes = [C.c_void_p, C.c_int32]
        L.nd_profile_read.argtypes = [C.c_void_p, C.POINTER(nd_profile)]
        L.nd_sweep_phases_get.argtypes = [C.c_void_p, C.c_void_p]
        L.nd_problem_info_get.argtypes = [C.c_void_p, C.POINTER(nd_problem_info)]
        L.nd_swath_stream_build.argtypes = [C.POINTER(nd_problem_desc), C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32,
                                            C.c_double, C.c_int32, C.POINTER(C.c_void_p)]
        L.nd_swath_stream_view.argtypes = [C.c_void_p, C.POINTER(nd_swath_stream_view_t)]
        L.nd_swath_stream_destroy.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _check(status, where, allow=()):
    if status != ND_OK and status not in allow:
        L = lib()
        raise NdError(L.nd_status_string(status).decode(), where, L.nd_last_error(None).decode())
    return status


def _ptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


def _np_view(addr, shape, dtype):
    n = int(np.prod(shape))
    if n == 0 or not addr:
        return np.zeros(shape, dtype)
    buf = (C.c_char * (n * np.dtype(dtype).itemsize)).from_address(addr)
    return np.frombuffer(buf, dtype=dtype).reshape(shape)


def nd_version():
    return int(lib().nd_version())


def nd_build_id():
    return lib().nd_build_id().decode()


class Tracks:
    """Result of nd_tracks_generate: numpy views of the library-owned host arrays (valid until .destroy()).
    Made by nd_tracks_generate_resident, the segment arrays live on the device (`seg_device`: the two device pointers, kept
    alive by `device_workspace`); `seg_region` / `seg_length` then copy them to the host on first use (nd_tracks_materialise)."""

    def __init__(self, handle, view, device_workspace=None, stream=None):
        self._h = handle
        T, R, S, NH = view.n_tracks, view.n_regions, view.n_segments, view.n_half
        self.n_tracks, self.n_regions, self.n_segments, self.n_half = T, R, S, NH
        self.seg_offset = _np_view(view.track_seg_offset, (T + 1,), np.int64)
        self.device_workspace, self._stream = device_workspace, stream
        self.seg_device = (int(view.seg_region_device), int(view.seg_length_device)) if view.seg_region_device else None
        self._seg_host = None
        if view.seg_region or S == 0:
            self._seg_host = (_np_view(view.seg_region, (S,), np.int32), _np_view(view.seg_length, (S,), np.float64))
        self.track_weight = _np_view(view.track_weight, (T,), np.float64)
        self.link = _np_view(view.link, (T, 2), np.int32)
        self.track_azim = _np_view(view.track_azim, (T,), np.int32)
        self.ends = _np_view(view.track_ends, (T, 4), np.float64)
        self.volume = _np_view(view.track_volume, (R,), np.float64)
        self.azim_phi = _np_view(view.azim_phi, (NH,), np.float64)
        self.azim_weight = _np_view(view.azim_weight, (NH,), np.float64)
        self.azim_spacing = _np_view(view.azim_spacing, (NH,), np.float64)
        self.track_global = _np_view(view.track_global, (T,), np.int32)
        self.is_shard = False

    def _materialise(self):
        if self._seg_host is None:
            _check(lib().nd_tracks_materialise(self._h, self._stream() if self._stream else None), "nd_tracks_materialise")
            v = nd_tracks_view_t()
            _check(lib().nd_tracks_view(self._h, C.byref(v)), "nd_tracks_view")
            self._seg_host = (_np_view(v.seg_region, (self.n_segments,), np.int32), _np_view(v.seg_length, (self.n_segments,), np.float64))
        return self._seg_host

    @property
    def on_host(self):
        return self._seg_host is not None

    @property
    def seg_region(self):
        return self._materialise()[0]

    @property
    def seg_length(self):
        return self._materialise()[1]

    def shard(self, n_shards, shard):
        """NEXT-2 (nd_tracks_shard): the tracks of one shard of the angle-pair partition, as a new Tracks object whose
        `volume` holds the areas of the WHOLE laydown and `track_global` the ids in this object."""
        self._materialise()
        h = C.c_void_p()
        _check(lib().nd_tracks_shard(self._h, int(n_shards), int(shard), C.byref(h)), "nd_tracks_shard")
        v = nd_tracks_view_t()
        _check(lib().nd_tracks_view(h, C.byref(v)), "nd_tracks_view")
        out = Tracks(h, v)
        out.is_shard = True
        return out

    def destroy(self):
        if self._h:
            lib().nd_tracks_destroy(self._h)
            self._h = None
        self.device_workspace = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def nd_tracks_generate(xy, tri, W, H, bc, n_azim, spacing, n_threads=0) -> Tracks:
    """Host preprocessing (row A0): cyclic track laydown + half-edge ray walk.  HOST arrays in, HOST views out."""
    xy = np.ascontiguousarray(xy, np.float64)
    tri = np.ascontiguousarray(tri, np.int32)
    md = nd_mesh_desc(len(xy), len(tri), xy.ctypes.data, tri.ctypes.data, float(W), float(H), (C.c_int32 * 4)(*[int(b) for b in bc]))
    h = C.c_void_p()
    _check(lib().nd_tracks_generate(C.byref(md), int(n_azim), float(spacing), int(n_threads), C.byref(h)), "nd_tracks_generate")
    v = nd_tracks_view_t()
    _check(lib().nd_tracks_view(h, C.byref(v)), "nd_tracks_view")
    return Tracks(h, v)


def nd_tracks_generate_device(xy, tri, W, H, bc, n_azim, spacing, segment_capacity=1 << 28, device="cuda:0") -> Tracks:
    """Row A0 with the ray walk on the GPU; bit-identical to nd_tracks_generate.  The torch
    workspace holds `segment_capacity` segments per fill batch (12 bytes each) and is released on return."""
    import torch
    xy = np.ascontiguousarray(xy, np.float64)
    tri = np.ascontiguousarray(tri, np.int32)
    md = nd_mesh_desc(len(xy), len(tri), xy.ctypes.data, tri.ctypes.data, float(W), float(H), (C.c_int32 * 4)(*[int(b) for b in bc]))
    nmin, per = C.c_size_t(), C.c_size_t()
    _check(lib().nd_tracks_device_workspace_bytes(C.byref(md), int(n_azim), float(spacing), C.byref(nmin), C.byref(per)),
           "nd_tracks_device_workspace_bytes")
    dev = torch.device(device)
    nbytes = int(nmin.value) + int(per.value) * int(segment_capacity)
    with torch.cuda.device(dev):
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)
        ptr = (ws.data_ptr() + 255) // 256 * 256
        h = C.c_void_p()
        tm = nd_trace_timing()
        _check(lib().nd_tracks_generate_device(C.byref(md), int(n_azim), float(spacing), C.c_void_p(ptr), nbytes,
                                               C.c_void_p(torch.cuda.current_stream(dev).cuda_stream), C.byref(tm), C.byref(h)),
               "nd_tracks_generate_device")
    del ws
    v = nd_tracks_view_t()
    _check(lib().nd_tracks_view(h, C.byref(v)), "nd_tracks_view")
    out = Tracks(h, v)
    out.timing = {f[0]: getattr(tm, f[0]) for f in nd_trace_timing._fields_ if f[0] != "reserved"}
    return out


def nd_tracks_generate_resident(xy, tri, W, H, bc, n_azim, spacing, segment_estimate=None, device="cuda:0") -> Tracks:
    """Row A0 on the GPU with the segments LEFT on the device (nd.h: nd_tracks_generate_resident).  The returned Tracks owns
    the torch workspace that holds them; pass it to nd_problem_create, which then builds its segment streams on the GPU.
    `segment_estimate` sizes the first attempt (default: Cauchy's mean-chord estimate, sum of the triangle perimeters /
    (pi * spacing) per angle, + 10 %); if the count pass finds more, the call is repeated once with the exact size."""
    import torch
    xy = np.ascontiguousarray(xy, np.float64)
    tri = np.ascontiguousarray(tri, np.int32)
    md = nd_mesh_desc(len(xy), len(tri), xy.ctypes.data, tri.ctypes.data, float(W), float(H), (C.c_int32 * 4)(*[int(b) for b in bc]))
    nmin, per = C.c_size_t(), C.c_size_t()
    _check(lib().nd_tracks_device_workspace_bytes(C.byref(md), int(n_azim), float(spacing), C.byref(nmin), C.byref(per)),
           "nd_tracks_device_workspace_bytes")
    if segment_estimate is None:
        p = xy[tri]
        perim = sum(np.hypot(*(p[:, (e + 1) % 3] - p[:, e]).T).sum() for e in range(3))
        segment_estimate = int(1.1 * (n_azim // 2) * perim / (np.pi * float(spacing))) + 4096
    dev = torch.device(device)
    nbytes = int(nmin.value) + int(per.value) * int(segment_estimate)
    stream = lambda: C.c_void_p(torch.cuda.current_stream(dev).cuda_stream)
    with torch.cuda.device(dev):
        for attempt in range(2):
            ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)
            ptr = (ws.data_ptr() + 255) // 256 * 256
            h, tm, need = C.c_void_p(), nd_trace_timing(), C.c_size_t(0)
            rc = lib().nd_tracks_generate_resident(C.byref(md), int(n_azim), float(spacing), C.c_void_p(ptr), nbytes, stream(),
                                                   C.byref(tm), C.byref(need), C.byref(h))
            if rc == ND_ERR_WORKSPACE and need.value > nbytes and attempt == 0:
                del ws
                nbytes = int(need.value)
                continue
            _check(rc, "nd_tracks_generate_resident")
            break
    v = nd_tracks_view_t()
    _check(lib().nd_tracks_view(h, C.byref(v)), "nd_tracks_view")
    out = Tracks(h, v, device_workspace=ws, stream=stream)
    out.timing = {f[0]: getattr(tm, f[0]) for f in nd_trace_timing._fields_ if f[0] != "reserved"}
    out.timing["attempts"] = attempt + 1
    return out


def nd_cmfd_surfaces(seg_offset, seg_region, link, cell, n_cells, n_regions=None):
    """C-2 (nd.h): the interior surfaces of the coarse mesh `cell` as sorted (pair_lo, pair_hi) int32 arrays.  HOST only."""
    so, sr = np.ascontiguousarray(seg_offset, np.int64), np.ascontiguousarray(seg_region, np.int32)
    lk, cell = np.ascontiguousarray(link, np.int32), np.ascontiguousarray(cell, np.int32)
    d = nd_problem_desc()
    d.n_regions, d.n_tracks = int(n_regions if n_regions is not None else len(cell)), len(so) - 1
    d.track_seg_offset, d.seg_region, d.link = so.ctypes.data, sr.ctypes.data, lk.ctypes.data
    n = C.c_int32()
    _check(lib().nd_cmfd_surfaces(C.byref(d), int(n_cells), cell.ctypes.data, 0, C.byref(n), None, None), "nd_cmfd_surfaces")
    lo, hi = np.empty(max(n.value, 1), np.int32), np.empty(max(n.value, 1), np.int32)
    if n.value:
        _check(lib().nd_cmfd_surfaces(C.byref(d), int(n_cells), cell.ctypes.data, n.value, C.byref(n), lo.ctypes.data,
                                      hi.ctypes.data), "nd_cmfd_surfaces")
    return lo[:n.value], hi[:n.value]


ND_STATIC_FISSION_MAX_ELEMENTS = 1 << 27


def nd_fission_rate_static(d_phi, d_region_material, d_nu_sigma_f, d_volume, d_out=None):
    """Allocation-free fission rate (nd.h): torch device tensors phi [R][G] f64, region_material [R] i32, nu_sigma_f [M][G] f64,
    volume [R] f64 in, a one-element f64 device tensor out (made here if not given: pass one to stay allocation-free)."""
    import torch
    R, G = d_phi.shape
    for t, dt in ((d_phi, torch.float64), (d_region_material, torch.int32), (d_nu_sigma_f, torch.float64), (d_volume, torch.float64)):
        assert t.is_cuda and t.is_contiguous() and t.dtype == dt
    assert d_region_material.numel() == R and d_volume.numel() == R and d_nu_sigma_f.shape[1] == G
    if d_out is None:
        d_out = torch.empty(1, dtype=torch.float64, device=d_phi.device)
    with torch.cuda.device(d_phi.device):
        _check(lib().nd_fission_rate_static(int(R), int(G), d_phi.data_ptr(), d_region_material.data_ptr(), d_nu_sigma_f.data_ptr(),
                                            d_volume.data_ptr(), d_out.data_ptr(),
                                            C.c_void_p(torch.cuda.current_stream(d_phi.device).cuda_stream)), "nd_fission_rate_static")
    return d_out


def nd_microbench(device="cuda:0", workspace_bytes=(1 << 30) + (2 << 20)):
    """Diagnostics (nd.h): MUFU.EX2 rate per clock per SM, SM clock, FP64 RED throughput (L2- / HBM-resident)."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        ws = torch.empty(int(workspace_bytes) + 256, dtype=torch.uint8, device=dev)
        ptr = (ws.data_ptr() + 255) // 256 * 256
        r = nd_microbench_result()
        _check(lib().nd_microbench(C.c_void_p(ptr), int(workspace_bytes), C.c_void_p(torch.cuda.current_stream(dev).cuda_stream),
                                   C.byref(r)), "nd_microbench")
    return {f[0]: getattr(r, f[0]) for f in nd_microbench_result._fields_ if f[0] != "reserved"}


class Problem:
    """Owner of an nd_problem handle and its torch workspace.  Methods mirror the C entry points."""

    def __init__(self, region_material, sigma_t, sigma_s, nu_sigma_f, chi, polar_sin, polar_weight, seg_offset,
                 seg_region, seg_length, track_weight, link, track_azim=None, track_ends=None, region_volume=None,
                 exp_mode=ND_EXP_FAST,
                 sweep_kernel=ND_SWEEP_AUTO, window_regions=0, block_warps=0, tile_segments=0,
                 delta_buffers=0, blocks_per_sm=0, tile_lag=0, q_copies=0, graph_mode=0, cmfd_stream=0, item_order=0, p1_stream=0, device="cuda:0",
                 seg_device=None):
        """seg_device = (device pointer of seg_region, of seg_length): the segments are device-resident
        (nd_problem_desc.seg_on_device = 1); seg_region / seg_length are then ignored and may be None."""
        import torch
        self.torch = torch
        self.device = torch.device(device)
        if seg_device is not None:
            seg_region, seg_length = np.zeros(0, np.int32), np.zeros(0, np.float64)
        keep = dict(
            rm=np.ascontiguousarray(region_material, np.int32), st=np.ascontiguousarray(sigma_t, np.float64),
            ss=np.ascontiguousarray(sigma_s, np.float64), nf=np.ascontiguousarray(nu_sigma_f, np.float64),
            ch=np.ascontiguousarray(chi, np.float64), ps=np.ascontiguousarray(polar_sin, np.float64),
            pw=np.ascontiguousarray(polar_weight, np.float64), so=np.ascontiguousarray(seg_offset, np.int64),
            sr=np.ascontiguousarray(seg_region, np.int32), sl=np.ascontiguousarray(seg_length, np.float64),
            tw=np.ascontiguousarray(track_weight, np.float64), lk=np.ascontiguousarray(link, np.int32))
        geo = [None, None]
        if track_azim is not None and track_ends is not None:
            keep["ta"] = np.ascontiguousarray(track_azim, np.int32)
            keep["te"] = np.ascontiguousarray(track_ends, np.float64)
            geo = [keep["ta"].ctypes.data, keep["te"].ctypes.data]
        if region_volume is not None:
            keep["rv"] = np.ascontiguousarray(region_volume, np.float64)
            geo = geo + [keep["rv"].ctypes.data]
        elif seg_device is not None:
            geo = geo + [None]
        self.R, (self.M, self.G), self.P, self.T = len(keep["rm"]), keep["st"].shape, len(keep["ps"]), len(keep["tw"])
        d = nd_problem_desc(self.R, self.M, self.G, self.P, self.T, *[keep[k].ctypes.data for k in
                            ("rm", "st", "ss", "nf", "ch", "ps", "pw", "so", "sr", "sl", "tw", "lk")], *geo)
        if seg_device is not None:
            d.seg_region, d.seg_length, d.seg_on_device = int(seg_device[0]), int(seg_device[1]), 1
        opt = nd_options(int(exp_mode), int(sweep_kernel), int(window_regions), int(block_warps),
                         int(tile_segments), int(delta_buffers), int(blocks_per_sm), int(tile_lag), int(q_copies), int(graph_mode), int(cmfd_stream), int(item_order), int(p1_stream))
        nbytes = C.c_size_t()
        _check(lib().nd_workspace_bytes(C.byref(d), C.byref(opt), C.byref(nbytes)), "nd_workspace_bytes")
        self.workspace_bytes = int(nbytes.value)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) // 256 * 256
            h = C.c_void_p()
            _check(lib().nd_problem_create(C.byref(d), C.byref(opt), C.c_void_p(self._ws_ptr), self.workspace_bytes,
                                           self._stream(), C.byref(h)), "nd_problem_create")
        self._h = h

    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def nd_problem_stream_view(self):
        """Diagnostics (nd.h): the swath kernel's chunk stream copied back from the workspace, as numpy arrays."""
        v = nd_stream_device_view_t()
        _check(lib().nd_problem_stream_view(self._h, C.byref(v)), "nd_problem_stream_view")
        base, t = self.workspace.data_ptr(), self.torch

        def grab(ptr, nbytes, dtype):
            off = int(ptr) - base
            return self.workspace[off:off + int(nbytes)].cpu().numpy().view(dtype)
        NT = v.tracks_per_swath
        return dict(blob=grab(v.blob, v.blob_bytes, np.uint8), tile_ref=grab(v.tile_ref, 8 * (v.n_tiles + 1), np.uint32).reshape(-1, 2),
                    swath_tile0=grab(v.swath_tile0, 8 * (v.n_swaths + 1), np.int64),
                    swath_track=grab(v.swath_track, 4 * v.n_swaths * NT, np.int32).reshape(-1, NT),
                    items=grab(v.items, 16 * v.n_items, np.int32).reshape(-1, 4), n_tiles=v.n_tiles, n_swaths=v.n_swaths,
                    tracks_per_swath=NT, built_on_device=bool(v.built_on_device))

    def nd_tally_reducer_set(self, fn):
        """NEXT-2 (nd.h): fn(tally) is called after every sweep with a torch FP64 tensor that ALIASES the problem's padded
        tally [R * Gs] and must replace it, in place and in stream order on the current stream, by the sum over the shards
        (e.g. torch.distributed.all_reduce).  fn = None removes the reducer."""
        if fn is None:
            self._reduce_cb = None
            _check(lib().nd_tally_reducer_set(self._h, C.cast(None, ND_TALLY_REDUCE_FN), None), "nd_tally_reducer_set")
            return
        t, base = self.torch, self.workspace.data_ptr()

        def cb(_user, ptr, n, _stream):
            try:
                off = int(ptr) - base
                fn(self.workspace[off:off + 8 * int(n)].view(t.float64))
                return 0
            except Exception:      # no exception may cross the C boundary
                import traceback
                traceback.print_exc()
                return 1
        self._reduce_cb = ND_TALLY_REDUCE_FN(cb)      # kept alive as long as the library may call it
        _check(lib().nd_tally_reducer_set(self._h, self._reduce_cb, None), "nd_tally_reducer_set")

    def destroy(self):
        if getattr(self, "_h", None):
            lib().nd_problem_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- compute entry points (device tensors in / out) ----
    def nd_transport_sweep(self, d_Q, d_phi_out=None):
        t = self.torch
        assert d_Q.dtype == t.float64 and d_Q.is_cuda and d_Q.is_contiguous() and d_Q.numel() == self.R * self.G
        if d_phi_out is None:
            d_phi_out = t.empty((self.R, self.G), dtype=t.float64, device=self.device)
        _check(lib().nd_transport_sweep(self._h, d_Q.data_ptr(), d_phi_out.data_ptr(), self._stream()), "nd_transport_sweep")
        return d_phi_out

    def nd_source_update(self, d_phi, k_eff, d_Q_out=None, want_fission_rate=False):
        t = self.torch
        assert d_phi.dtype == t.float64 and d_phi.is_cuda and d_phi.is_contiguous() and d_phi.numel() == self.R * self.G
        if d_Q_out is None:
            d_Q_out = t.empty((self.R, self.G), dtype=t.float64, device=self.device)
        d_F = t.empty(1, dtype=t.float64, device=self.device) if want_fission_rate else None
        _check(lib().nd_source_update(self._h, d_phi.data_ptr(), float(k_eff), d_Q_out.data_ptr(),
                                      d_F.data_ptr() if d_F is not None else None, self._stream()), "nd_source_update")
        return (d_Q_out, d_F) if want_fission_rate else d_Q_out

    def nd_power_iteration(self, max_iters, tol_k=0.0, tol_phi=0.0, d_phi_out=None, want_stats=False):
        k = C.c_double()
        it = C.c_int32()
        stats = (nd_iter_stats * max(1, max_iters))() if want_stats else None
        rc = lib().nd_power_iteration(self._h, int(max_iters), float(tol_k), float(tol_phi), C.byref(k),
                                      d_phi_out.data_ptr() if d_phi_out is not None else None, C.byref(it),
                                      C.cast(stats, C.c_void_p) if stats is not None else None, self._stream())
        _check(rc, "nd_power_iteration", allow=(ND_ERR_NOT_CONVERGED,))
        out = dict(k_eff=k.value, iters=it.value, converged=(rc == ND_OK))
        if want_stats:
            out["stats"] = [dict(k_eff=s.k_eff, fission_rate=s.fission_rate, dk=s.dk, dphi_max=s.dphi_max, leakage=s.leakage,
                                 balance_residual=s.balance_residual) for s in stats[:it.value]]
        return out

    # ---- state ----
    def nd_state_reset(self):
        _check(lib().nd_state_reset(self._h, self._stream()), "nd_state_reset")

    def nd_boundary_flux_fill(self, value):
        _check(lib().nd_boundary_flux_fill(self._h, float(value), self._stream()), "nd_boundary_flux_fill")

    def nd_boundary_flux_get(self):
        out = np.empty((self.T, 2, self.P, self.G), np.float32)
        _check(lib().nd_boundary_flux_get(self._h, out.ctypes.data, self._stream()), "nd_boundary_flux_get")
        return out

    def nd_outgoing_flux_get(self):
        out = np.empty((self.T, 2, self.P, self.G), np.float32)
        _check(lib().nd_outgoing_flux_get(self._h, out.ctypes.data, self._stream()), "nd_outgoing_flux_get")
        return out

    def nd_boundary_flux_set(self, psi):
        psi = np.ascontiguousarray(psi, np.float32)
        assert psi.size == self.T * 2 * self.P * self.G
        _check(lib().nd_boundary_flux_set(self._h, psi.ctypes.data, self._stream()), "nd_boundary_flux_set")

    def nd_flux_get(self):
        out = self.torch.empty((self.R, self.G), dtype=self.torch.float64, device=self.device)
        _check(lib().nd_flux_get(self._h, out.data_ptr(), self._stream()), "nd_flux_get")
        return out

    def nd_flux_set(self, d_phi, k_eff):
        _check(lib().nd_flux_set(self._h, d_phi.data_ptr(), float(k_eff), self._stream()), "nd_flux_set")

    def nd_track_volume_get(self):
        out = np.empty(self.R, np.float64)
        _check(lib().nd_track_volume_get(self._h, out.ctypes.data), "nd_track_volume_get")
        return out

    def nd_tally_get(self):
        out = self.torch.empty((self.R, self.G), dtype=self.torch.float64, device=self.device)
        _check(lib().nd_tally_get(self._h, out.data_ptr(), self._stream()), "nd_tally_get")
        return out

    def nd_cmfd_create(self, seg_offset, seg_region, link, cell, n_cells, pair_lo, pair_hi, coupling, tol=0.0, max_outer=0,
                       inner_sweeps=0, relax=0.0, rel_tol=0.0):
        """NEXT-3 (nd.h): a CMFD plan on this problem.  seg_offset / seg_region / link: the arrays the problem was created from."""
        return Cmfd(self, seg_offset, seg_region, link, cell, n_cells, pair_lo, pair_hi, coupling, tol, max_outer, inner_sweeps, relax,
                    rel_tol)

    def nd_profile_enable(self, on=True):
        _check(lib().nd_profile_enable(self._h, int(on)), "nd_profile_enable")

    def nd_sweep_phases_get(self):
        out = np.zeros(6, np.float64)
        _check(lib().nd_sweep_phases_get(self._h, out.ctypes.data), "nd_sweep_phases_get")
        return dict(zip(("stage", "wait_before_loop", "segment_loop", "wait_after_loop", "flush", "between_tiles"), out.tolist()))

    def nd_profile_read(self):
        pr = nd_profile()
        _check(lib().nd_profile_read(self._h, C.byref(pr)), "nd_profile_read")
        return dict(sweep_ms=pr.sweep_ms, sweep_launches=pr.sweep_launches, kernels_launched=pr.kernels_launched)

    def nd_problem_info_get(self):
        inf = nd_problem_info()
        _check(lib().nd_problem_info_get(self._h, C.byref(inf)), "nd_problem_info_get")
        return {f[0]: getattr(inf, f[0]) for f in nd_problem_info._fields_ if f[0] != "reserved"}


class P1:
    """Owner of an nd_p1 plan and its torch workspace (include/nd.h "NEXT-4": P_1 scattering source).  tracks: the Tracks (or
    any object with seg_offset, seg_region, seg_length, track_weight, ends) the problem was created from."""

    def __init__(self, prob, tracks, polar_sin, polar_weight, sigma_s1):
        t = prob.torch
        self.prob = prob
        keep = dict(so=np.ascontiguousarray(tracks.seg_offset, np.int64), sr=np.ascontiguousarray(tracks.seg_region, np.int32),
                    sl=np.ascontiguousarray(tracks.seg_length, np.float64), tw=np.ascontiguousarray(tracks.track_weight, np.float64),
                    te=np.ascontiguousarray(tracks.ends, np.float64), ps=np.ascontiguousarray(polar_sin, np.float64),
                    pw=np.ascontiguousarray(polar_weight, np.float64), s1=np.ascontiguousarray(sigma_s1, np.float64))
        assert keep["s1"].shape == (prob.M, prob.G, prob.G)
        d = nd_problem_desc()
        d.n_regions, d.n_tracks, d.n_polar = prob.R, prob.T, prob.P
        d.track_seg_offset, d.seg_region, d.seg_length = keep["so"].ctypes.data, keep["sr"].ctypes.data, keep["sl"].ctypes.data
        d.track_weight, d.track_ends = keep["tw"].ctypes.data, keep["te"].ctypes.data
        d.polar_sin, d.polar_weight = keep["ps"].ctypes.data, keep["pw"].ctypes.data
        nbytes = C.c_size_t()
        _check(lib().nd_p1_workspace_bytes(prob._h, C.byref(nbytes)), "nd_p1_workspace_bytes")
        with t.cuda.device(prob.device):
            self.workspace = t.empty(int(nbytes.value) + 256, dtype=t.uint8, device=prob.device)
            ptr = (self.workspace.data_ptr() + 255) // 256 * 256
            h = C.c_void_p()
            _check(lib().nd_p1_create(prob._h, C.byref(d), keep["s1"].ctypes.data, C.c_void_p(ptr), int(nbytes.value), prob._stream(),
                                      C.byref(h)), "nd_p1_create")
        self._h = h

    def destroy(self):
        if getattr(self, "_h", None):
            lib().nd_p1_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def _new(self):
        t = self.prob.torch
        return t.empty((self.prob.R, self.prob.G), dtype=t.float64, device=self.prob.device)

    def nd_p1_transport_sweep(self, d_Q0, d_Q1x, d_Q1y):
        phi, Jx, Jy = self._new(), self._new(), self._new()
        _check(lib().nd_p1_transport_sweep(self._h, d_Q0.data_ptr(), d_Q1x.data_ptr(), d_Q1y.data_ptr(), phi.data_ptr(), Jx.data_ptr(),
                                           Jy.data_ptr(), self.prob._stream()), "nd_p1_transport_sweep")
        return phi, Jx, Jy

    def nd_p1_source_update(self, d_phi, d_Jx, d_Jy, k_eff):
        Q0, Q1x, Q1y = self._new(), self._new(), self._new()
        _check(lib().nd_p1_source_update(self._h, d_phi.data_ptr(), d_Jx.data_ptr(), d_Jy.data_ptr(), float(k_eff), Q0.data_ptr(),
                                         Q1x.data_ptr(), Q1y.data_ptr(), self.prob._stream()), "nd_p1_source_update")
        return Q0, Q1x, Q1y

    def nd_p1_state_reset(self):
        _check(lib().nd_p1_state_reset(self._h, self.prob._stream()), "nd_p1_state_reset")

    def nd_p1_power_iteration(self, n_iters):
        k = C.c_double()
        phi, Jx, Jy = self._new(), self._new(), self._new()
        hist = np.empty(max(1, n_iters))
        _check(lib().nd_p1_power_iteration(self._h, int(n_iters), C.byref(k), phi.data_ptr(), Jx.data_ptr(), Jy.data_ptr(),
                                           hist.ctypes.data, self.prob._stream()), "nd_p1_power_iteration")
        return dict(k_eff=k.value, phi=phi, Jx=Jx, Jy=Jy, k_history=hist[:n_iters])


class Cmfd:
    """Owner of an nd_cmfd plan and its torch workspace (include/nd.h "NEXT-3").  Methods mirror the C entry points."""

    def __init__(self, prob, seg_offset, seg_region, link, cell, n_cells, pair_lo, pair_hi, coupling, tol, max_outer,
                 inner_sweeps, relax, rel_tol=0.0):
        t = prob.torch
        self.prob, self.n_cells, self.G = prob, int(n_cells), prob.G
        keep = dict(so=np.ascontiguousarray(seg_offset, np.int64), sr=np.ascontiguousarray(seg_region, np.int32),
                    lk=np.ascontiguousarray(link, np.int32), cell=np.ascontiguousarray(cell, np.int32),
                    lo=np.ascontiguousarray(pair_lo, np.int32), hi=np.ascontiguousarray(pair_hi, np.int32),
                    cp=np.ascontiguousarray(coupling, np.float64))
        assert keep["cell"].shape == (prob.R,) and keep["lo"].shape == keep["hi"].shape == keep["cp"].shape
        self.n_pairs = len(keep["lo"])
        d = nd_problem_desc()
        d.n_regions, d.n_tracks = prob.R, prob.T
        d.track_seg_offset, d.seg_region, d.link = keep["so"].ctypes.data, keep["sr"].ctypes.data, keep["lk"].ctypes.data
        nbytes = C.c_size_t()
        _check(lib().nd_cmfd_workspace_bytes(prob._h, C.byref(d), self.n_cells, keep["cell"].ctypes.data, self.n_pairs,
                                             C.byref(nbytes)), "nd_cmfd_workspace_bytes")
        opt = nd_cmfd_options(float(tol), int(max_outer), int(inner_sweeps), float(relax), float(rel_tol))
        with t.cuda.device(prob.device):
            self.workspace = t.empty(int(nbytes.value) + 256, dtype=t.uint8, device=prob.device)
            ptr = (self.workspace.data_ptr() + 255) // 256 * 256
            h = C.c_void_p()
            _check(lib().nd_cmfd_create(prob._h, C.byref(d), self.n_cells, keep["cell"].ctypes.data, self.n_pairs,
                                        keep["lo"].ctypes.data, keep["hi"].ctypes.data, keep["cp"].ctypes.data, C.byref(opt),
                                        C.c_void_p(ptr), int(nbytes.value), prob._stream(), C.byref(h)), "nd_cmfd_create")
        self._h = h

    def destroy(self):
        if getattr(self, "_h", None):
            lib().nd_cmfd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def nd_cmfd_iteration(self, n_iters, want_stats=False):
        k = C.c_double()
        stats = (nd_cmfd_stats * max(1, n_iters))() if want_stats else None
        _check(lib().nd_cmfd_iteration(self._h, int(n_iters), C.byref(k), C.cast(stats, C.c_void_p) if stats is not None else None,
                                       self.prob._stream()), "nd_cmfd_iteration")
        out = dict(k_eff=k.value)
        if want_stats:
            out["stats"] = [dict(k_sweep=s.k_sweep, k_eff=s.k_eff, coarse_iters=s.coarse_iters, coarse_ok=s.coarse_ok)
                            for s in stats[:n_iters]]
        return out

    def nd_cmfd_sweep(self, d_Q, d_phi_out=None):
        t = self.prob.torch
        assert d_Q.dtype == t.float64 and d_Q.is_cuda and d_Q.is_contiguous() and d_Q.numel() == self.prob.R * self.G
        if d_phi_out is None:
            d_phi_out = t.empty((self.prob.R, self.G), dtype=t.float64, device=self.prob.device)
        _check(lib().nd_cmfd_sweep(self._h, d_Q.data_ptr(), d_phi_out.data_ptr(), self.prob._stream()), "nd_cmfd_sweep")
        return d_phi_out

    def nd_cmfd_currents_get(self):
        Js, Jv, Jr = np.empty((self.n_pairs, self.G)), np.empty((self.n_cells, self.G)), np.empty((self.n_cells, self.G))
        _check(lib().nd_cmfd_currents_get(self._h, Js.ctypes.data, Jv.ctypes.data, Jr.ctypes.data, self.prob._stream()),
               "nd_cmfd_currents_get")
        return Js, Jv, Jr

    def nd_cmfd_collapse(self, d_phi=None):
        _check(lib().nd_cmfd_collapse(self._h, d_phi.data_ptr() if d_phi is not None else None, self.prob._stream()), "nd_cmfd_collapse")

    def nd_cmfd_coarse_get(self):
        n, G = self.n_cells, self.G
        out = dict(V=np.empty(n), Phi=np.empty((n, G)), sigt=np.empty((n, G)), sigs=np.empty((n, G, G)), nusf=np.empty((n, G)),
                   chi=np.empty((n, G)))
        _check(lib().nd_cmfd_coarse_get(self._h, out["V"].ctypes.data, out["Phi"].ctypes.data, out["sigt"].ctypes.data,
                                        out["sigs"].ctypes.data, out["nusf"].ctypes.data, out["chi"].ctypes.data,
                                        self.prob._stream()), "nd_cmfd_coarse_get")
        return out

    def nd_cmfd_coarse_set(self, co, J_surf, J_vac):
        f8 = lambda a: np.ascontiguousarray(a, np.float64)
        V, Phi, st, ss, nf, ch, Js, Jv = (f8(a) for a in (co["V"], co["Phi"], co["sigt"], co["sigs"], co["nusf"], co["chi"], J_surf, J_vac))
        n, G = self.n_cells, self.G
        assert Phi.shape == (n, G) and ss.shape == (n, G, G) and Js.shape == (self.n_pairs, G) and Jv.shape == (n, G)
        _check(lib().nd_cmfd_coarse_set(self._h, V.ctypes.data, Phi.ctypes.data, st.ctypes.data, ss.ctypes.data, nf.ctypes.data,
                                        ch.ctypes.data, Js.ctypes.data, Jv.ctypes.data, self.prob._stream()), "nd_cmfd_coarse_set")

    def nd_cmfd_solve(self, k0, allow=()):
        k, it, out = C.c_double(), C.c_int32(), np.empty((self.n_cells, self.G))
        rc = lib().nd_cmfd_solve(self._h, float(k0), C.byref(k), out.ctypes.data, C.byref(it), self.prob._stream())
        _check(rc, "nd_cmfd_solve", allow=allow)
        return k.value, out, it.value, rc

    def nd_cmfd_prolong(self):
        _check(lib().nd_cmfd_prolong(self._h, self.prob._stream()), "nd_cmfd_prolong")


def nd_swath_stream_build(region_material, n_materials, seg_offset, seg_region, seg_length, tracks_per_swath,
                          tile_segments, window_regions, slots_per_line, row_bytes, track_azim=None, track_ends=None,
                          lag_segments=-1.0, item_order=0):
    """Diagnostics (HOST only, no GPU): the swath/tile chunk stream of ND_SWEEP_SWATH as numpy copies.
    Returns a dict with blob (uint8), tile_ref [n_tiles+1][2], swath_tile0, swath_track [n_swaths][NT], items [n][4] and stats."""
    keep = dict(rm=np.ascontiguousarray(region_material, np.int32), so=np.ascontiguousarray(seg_offset, np.int64),
                sr=np.ascontiguousarray(seg_region, np.int32), sl=np.ascontiguousarray(seg_length, np.float64))
    d = nd_problem_desc()
    d.n_regions, d.n_materials, d.n_groups, d.n_polar, d.n_tracks = len(keep["rm"]), int(n_materials), 1, 1, len(keep["so"]) - 1
    d.region_material, d.track_seg_offset = keep["rm"].ctypes.data, keep["so"].ctypes.data
    d.seg_region, d.seg_length = keep["sr"].ctypes.data, keep["sl"].ctypes.data
    if track_azim is not None and track_ends is not None:
        keep["ta"] = np.ascontiguousarray(track_azim, np.int32)
        keep["te"] = np.ascontiguousarray(track_ends, np.float64)
        d.track_azim, d.track_ends = keep["ta"].ctypes.data, keep["te"].ctypes.data
    h = C.c_void_p()
    _check(lib().nd_swath_stream_build(C.byref(d), int(tracks_per_swath), int(tile_segments), int(window_regions),
                                       int(slots_per_line), int(row_bytes), float(lag_segments), int(item_order), C.byref(h)),
               "nd_swath_stream_build")
    try:
        v = nd_swath_stream_view_t()
        _check(lib().nd_swath_stream_view(h, C.byref(v)), "nd_swath_stream_view")
        return dict(n_swaths=v.n_swaths, n_tiles=v.n_tiles,
                    blob=_np_view(v.blob, (v.blob_bytes,), np.uint8).copy(),
                    tile_ref=_np_view(v.tile_ref, (v.n_tiles + 1, 2), np.uint32).copy(),
                    swath_tile0=_np_view(v.swath_tile0, (v.n_swaths + 1,), np.int64).copy(),
                    swath_track=_np_view(v.swath_track, (v.n_swaths, int(tracks_per_swath)), np.int32).copy(),
                    items=_np_view(v.items, (v.n_items, 4), np.int32).copy(),
                    mean_regions_per_tile=v.mean_regions_per_tile, mean_segments_per_tile=v.mean_segments_per_tile,
                    lockstep_efficiency=v.lockstep_efficiency, max_head_bytes=v.max_head_bytes, max_rec_bytes=v.max_rec_bytes)
    finally:
        lib().nd_swath_stream_destroy(h)


def nd_problem_create(xs, polar_sin, polar_weight, region_material, tracks, **options) -> Problem:
    """Convenience: build a Problem from a cross-section set (arrays sigma_t, sigma_s, nu_sigma_f, chi) and Tracks."""
    host_build = options.pop("host_build", False)       # device-resident tracks: materialise them and use the host builder
    resident = getattr(tracks, "seg_device", None) is not None and not host_build
    return Problem(region_material, xs.sigma_t, xs.sigma_s, xs.nu_sigma_f, xs.chi, polar_sin, polar_weight,
                   tracks.seg_offset, None if resident else tracks.seg_region, None if resident else tracks.seg_length,
                   tracks.track_weight, tracks.link, track_azim=tracks.track_azim, track_ends=tracks.ends,
                   seg_device=tracks.seg_device if resident else None,
                   region_volume=getattr(tracks, "volume", None), **options)     # the library's own A~_r (whole laydown for a shard)
