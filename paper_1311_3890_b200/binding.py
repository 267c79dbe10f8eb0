"""Thin ctypes binding of libtbsma.so (include/tbsma.h): argument marshalling only.

Same names as the C ABI (`tbsma_*` -> methods of `Context`).  PyTorch supplies device memory
and streams, nothing else: every step of the path runs in the library's CUDA kernels.  There is
no CPU fallback -- if the library is missing or no CUDA device exists this module raises.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtbsma.so")

OK, EINVAL, ENOMEM, ECUDA, ESTATE, ELIMIT = 0, -1, -2, -3, -4, -5
NOALLOC_MAX_REPLICAS = 4096          # TBSMA_NOALLOC_MAX_REPLICAS of tbsma.h
FLAG_NLIST_OVERFLOW, FLAG_OUT_OF_BOX, FLAG_NONFINITE, FLAG_SKIN_VIOLATED, FLAG_TILE_OVERFLOW = 1, 2, 4, 8, 16

EXPORTS = [
    "tbsma_create", "tbsma_destroy", "tbsma_set_system", "tbsma_build_cells", "tbsma_build_neighbors",
    "tbsma_compute", "tbsma_md_step", "tbsma_md_run", "tbsma_md_run_host", "tbsma_get_neighbors",
    "tbsma_count_pairs", "tbsma_kinetic_tensor", "tbsma_kinetic_tensor_noalloc", "tbsma_stress", "tbsma_status", "tbsma_clear_status", "tbsma_get_stats", "tbsma_set_variant",
    "tbsma_get_variant", "tbsma_get_tiling", "tbsma_set_tile", "tbsma_set_overlap", "tbsma_set_stagger", "tbsma_set_thermostat", "tbsma_get_thermostat", "tbsma_set_thermostat_state", "tbsma_set_async", "tbsma_set_balance", "tbsma_set_outer_skin", "tbsma_set_tile_split", "tbsma_set_gather", "tbsma_set_tile_box", "tbsma_set_fused_step", "tbsma_get_fused_step",
    "tbsma_set_protocol", "tbsma_set_series", "tbsma_series_histogram",
    "tbsma_set_graph", "tbsma_set_timing", "tbsma_get_timing", "tbsma_launch_count", "tbsma_strerror", "tbsma_version",
]


class Params(C.Structure):
    _fields_ = [("A", C.c_double), ("xi", C.c_double), ("p", C.c_double), ("q", C.c_double),
                ("r0", C.c_double), ("mass_amu", C.c_double)]


class Stats(C.Structure):
    _fields_ = [("n_steps", C.c_uint64), ("n_replica_builds", C.c_uint64), ("n_build_passes", C.c_uint64),
                ("max_neighbors_seen", C.c_int32), ("n_candidate_builds", C.c_int32)]


class Protocol(C.Structure):
    _fields_ = [("d_slab1_disp0", C.c_void_p), ("d_slab1_rate", C.c_void_p), ("stepwise_period", C.c_int64),
                ("d_T_rate", C.c_void_p)]


class Series(C.Structure):
    _fields_ = [("every", C.c_int32), ("capacity", C.c_int32), ("d_series", C.c_void_p), ("d_count", C.c_void_p),
                ("d_rupture_step", C.c_void_p), ("d_volume", C.c_void_p), ("d_L0", C.c_void_p)]


def au_params():
    """Table 1 of the paper, r0 = a/sqrt(2) (reading A1), Au mass."""
    return Params(0.2061, 1.790, 10.229, 4.036, 2.884, 196.96657)


class TbsmaError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"{what}: {code} ({strerror(code)})")
        self.code = code


_lib = None


def lib():
    """Load libtbsma.so; loud failure if it has not been built (python -m paper_1311_3890_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1311_3890_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        L.tbsma_create.argtypes = [C.POINTER(Params), dbl, dbl, C.POINTER(vp)]
        L.tbsma_destroy.argtypes = [vp]
        L.tbsma_set_system.argtypes = [vp, i64, i32, vp, vp, vp, vp, i32]
        L.tbsma_build_cells.argtypes = [vp, vp, vp, vp, vp]
        L.tbsma_build_neighbors.argtypes = [vp, vp, vp, vp, vp]
        L.tbsma_compute.argtypes = [vp, vp, vp, vp, vp, vp]
        L.tbsma_md_step.argtypes = [vp, vp, vp, vp, vp, dbl, vp, dbl, vp, C.c_uint64, vp, vp, vp, vp, vp]
        L.tbsma_md_run.argtypes = [vp, vp, vp, vp, vp, dbl, vp, dbl, vp, C.c_uint64, i64, vp, vp, i32, vp, vp, vp, vp]
        L.tbsma_md_run_host.argtypes = [vp, vp, vp, vp, vp, dbl, vp, dbl, vp, C.c_uint64, i64, vp, vp, i32, vp, vp, vp]
        L.tbsma_get_neighbors.argtypes = [vp, vp, vp, vp, vp]
        L.tbsma_kinetic_tensor.argtypes = [vp, vp, vp, vp, vp]
        L.tbsma_kinetic_tensor_noalloc.argtypes = [vp, vp, vp, i64, i32, dbl, vp, vp]
        L.tbsma_stress.argtypes = [vp, vp, vp, vp, vp, vp]
        L.tbsma_count_pairs.argtypes = [vp, vp, C.POINTER(i64), C.POINTER(i64), vp]
        L.tbsma_status.argtypes = [vp, C.POINTER(C.c_uint32)]
        L.tbsma_clear_status.argtypes = [vp]
        L.tbsma_get_stats.argtypes = [vp, C.POINTER(Stats)]
        L.tbsma_set_variant.argtypes = [vp, i32]
        L.tbsma_get_variant.argtypes = [vp]
        L.tbsma_set_tile.argtypes = [vp, i32, i32]
        L.tbsma_set_graph.argtypes = [vp, i32]
        L.tbsma_set_overlap.argtypes = [vp, i32]
        L.tbsma_set_stagger.argtypes = [vp, i32]
        L.tbsma_set_thermostat.argtypes = [vp, i32, dbl]
        L.tbsma_get_thermostat.argtypes = [vp, vp, vp]
        L.tbsma_set_thermostat_state.argtypes = [vp, vp, vp]
        L.tbsma_set_async.argtypes = [vp, i32, dbl]
        L.tbsma_set_balance.argtypes = [vp, i32, dbl]
        L.tbsma_set_outer_skin.argtypes = [vp, dbl]
        L.tbsma_set_tile_split.argtypes = [vp, i32]
        L.tbsma_set_gather.argtypes = [vp, i32]
        L.tbsma_set_fused_step.argtypes = [vp, i32]
        L.tbsma_get_fused_step.argtypes = [vp]
        L.tbsma_get_tiling.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32)]
        L.tbsma_set_tile_box.argtypes = [vp, i32]
        L.tbsma_set_protocol.argtypes = [vp, C.POINTER(Protocol)]
        L.tbsma_set_series.argtypes = [vp, C.POINTER(Series)]
        L.tbsma_series_histogram.argtypes = [vp, vp, vp, i32, i32, i32, dbl, dbl, i32, dbl, dbl, i32, vp, vp]
        L.tbsma_set_timing.argtypes = [vp, i32]
        L.tbsma_get_timing.argtypes = [vp, C.POINTER(dbl), C.POINTER(i64)]
        L.tbsma_launch_count.argtypes = [vp]
        L.tbsma_launch_count.restype = i64
        L.tbsma_strerror.argtypes = [C.c_int]
        L.tbsma_strerror.restype = C.c_char_p
        L.tbsma_version.restype = C.c_char_p
        _lib = L
    return _lib


def strerror(code):
    return lib().tbsma_strerror(int(code)).decode()


def version():
    return lib().tbsma_version().decode()


def _dp(t):
    """device pointer of a torch tensor (or None)"""
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "expected a contiguous CUDA tensor"
    return C.c_void_p(t.data_ptr())


def _hp(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _check(rc, what):
    if rc != 0:
        raise TbsmaError(rc, what)


def kinetic_tensor_noalloc(pos, vel, replica_offsets, k_rep, mass_amu=None, stream=None):
    """tbsma_kinetic_tensor_noalloc: the kinetic tensor of every replica without a Context and without any device
    allocation by the library -- for a caller that lives inside somebody else's memory pool, or between the steps of a loop
    that cannot take the device-wide stall of a cudaMalloc.  All four tensors are the caller's CUDA tensors:
    pos, vel (n x 4 float32), replica_offsets (R + 1 int32, ON THE DEVICE), k_rep (R x 6 float64, overwritten).  The
    library's working memory is one fixed array per GPU shared by every call: at most NOALLOC_MAX_REPLICAS replicas
    (TbsmaError with code ELIMIT beyond), and calls must not overlap on the GPU (same stream, or ordered by events).
    Make the first call on a GPU outside any stream capture."""
    assert replica_offsets.dtype == torch.int32 and k_rep.dtype == torch.float64
    n, R = int(pos.shape[0]), int(replica_offsets.numel()) - 1
    m = au_params().mass_amu if mass_amu is None else float(mass_amu)
    _check(lib().tbsma_kinetic_tensor_noalloc(_dp(pos), _dp(vel), _dp(replica_offsets), n, R, m, _dp(k_rep),
                                              _stream(stream)), "tbsma_kinetic_tensor_noalloc")


class Context:
    """One tbsma_ctx.  Methods mirror the C entry points one to one."""

    def __init__(self, params=None, r_cut=7.0, skin=0.3):
        self.params = params or au_params()
        self._h = C.c_void_p()
        _check(lib().tbsma_create(C.byref(self.params), r_cut, skin, C.byref(self._h)), "tbsma_create")
        self.n = 0
        self.R = 0
        self.max_neighbors = 0

    def destroy(self):
        if self._h:
            lib().tbsma_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def set_system(self, offsets, box_lo, box_hi, periodic, max_neighbors=112):
        offsets = np.ascontiguousarray(offsets, dtype=np.int32)
        R = len(offsets) - 1
        lo = np.ascontiguousarray(np.broadcast_to(np.asarray(box_lo, np.float32), (R, 3)))
        hi = np.ascontiguousarray(np.broadcast_to(np.asarray(box_hi, np.float32), (R, 3)))
        per = np.ascontiguousarray(np.broadcast_to(np.asarray(periodic, np.uint8), (R, 3)))
        _check(lib().tbsma_set_system(self._h, int(offsets[-1]), R, _hp(offsets), _hp(lo), _hp(hi), _hp(per),
                                      int(max_neighbors)), "tbsma_set_system")
        self.n, self.R = int(offsets[-1]), R
        self.max_neighbors = (int(max_neighbors) + 3) // 4 * 4

    def build_cells(self, pos, vel, tag, stream=None):
        _check(lib().tbsma_build_cells(self._h, _dp(pos), _dp(vel), _dp(tag), _stream(stream)), "tbsma_build_cells")

    def build_neighbors(self, pos, vel, tag, stream=None):
        _check(lib().tbsma_build_neighbors(self._h, _dp(pos), _dp(vel), _dp(tag), _stream(stream)),
               "tbsma_build_neighbors")

    def compute(self, pos, force_energy, replica_energy=None, replica_virial=None, stream=None):
        _check(lib().tbsma_compute(self._h, _dp(pos), _dp(force_energy), _dp(replica_energy), _dp(replica_virial),
                                   _stream(stream)), "tbsma_compute")

    def md_step(self, pos, vel, force_energy, tag, dt_fs, T, gamma_per_fs, seed, step, slab_disp=None,
                replica_energy=None, replica_virial=None, replica_ekin=None, stream=None):
        _check(lib().tbsma_md_step(self._h, _dp(pos), _dp(vel), _dp(force_energy), _dp(tag), float(dt_fs), _dp(T),
                                   float(gamma_per_fs), _dp(seed), int(step), _dp(slab_disp), _dp(replica_energy),
                                   _dp(replica_virial), _dp(replica_ekin), _stream(stream)), "tbsma_md_step")

    def md_run(self, pos, vel, force_energy, tag, dt_fs, T, gamma_per_fs, seed, step0, n_steps, slab_disp0=None,
               slab_rate=None, rebuild_every=0, replica_energy=None, replica_virial=None, replica_ekin=None,
               stream=None):
        _check(lib().tbsma_md_run(self._h, _dp(pos), _dp(vel), _dp(force_energy), _dp(tag), float(dt_fs), _dp(T),
                                  float(gamma_per_fs), _dp(seed), int(step0), int(n_steps), _dp(slab_disp0),
                                  _dp(slab_rate), int(rebuild_every), _dp(replica_energy), _dp(replica_virial),
                                  _dp(replica_ekin), _stream(stream)), "tbsma_md_run")

    def md_run_host(self, pos, vel, force_energy, tag, dt_fs, T, gamma_per_fs, seed, step0, n_steps,
                    slab_disp0=None, slab_rate=None, rebuild_every=0, replica_energy=None, replica_virial=None,
                    replica_ekin=None):
        """HOST numpy buffers in/out (pos, vel, force_energy: (n,4) float32; tag: (n,) int32)."""
        _check(lib().tbsma_md_run_host(self._h, _hp(pos), _hp(vel), _hp(force_energy), _hp(tag), float(dt_fs),
                                       _hp(T), float(gamma_per_fs), _hp(seed), int(step0), int(n_steps),
                                       _hp(slab_disp0), _hp(slab_rate), int(rebuild_every), _hp(replica_energy),
                                       _hp(replica_virial), _hp(replica_ekin)), "tbsma_md_run_host")

    def kinetic_tensor(self, pos, vel, k_rep, stream=None):
        _check(lib().tbsma_kinetic_tensor(self._h, _dp(pos), _dp(vel), _dp(k_rep), _stream(stream)), "tbsma_kinetic_tensor")

    def stress(self, w_rep, k_rep, volume, sigma, stream=None):
        _check(lib().tbsma_stress(self._h, _dp(w_rep), _dp(k_rep), _dp(volume), _dp(sigma), _stream(stream)), "tbsma_stress")

    def get_neighbors(self, tag, counts, nlist, stream=None):
        _check(lib().tbsma_get_neighbors(self._h, _dp(tag), _dp(counts), _dp(nlist), _stream(stream)),
               "tbsma_get_neighbors")

    def count_pairs(self, pos, stream=None):
        a, b = C.c_int64(0), C.c_int64(0)
        _check(lib().tbsma_count_pairs(self._h, _dp(pos), C.byref(a), C.byref(b), _stream(stream)), "tbsma_count_pairs")
        return int(a.value), int(b.value)

    def status(self):
        f = C.c_uint32(0)
        _check(lib().tbsma_status(self._h, C.byref(f)), "tbsma_status")
        return int(f.value)

    def clear_status(self):
        _check(lib().tbsma_clear_status(self._h), "tbsma_clear_status")

    def get_stats(self):
        s = Stats()
        _check(lib().tbsma_get_stats(self._h, C.byref(s)), "tbsma_get_stats")
        return dict(n_steps=int(s.n_steps), n_replica_builds=int(s.n_replica_builds),
                    n_build_passes=int(s.n_build_passes), max_neighbors_seen=int(s.max_neighbors_seen),
                    n_candidate_builds=int(s.n_candidate_builds))

    def set_variant(self, variant):
        _check(lib().tbsma_set_variant(self._h, int(variant)), "tbsma_set_variant")

    def get_variant(self):
        return int(lib().tbsma_get_variant(self._h))

    def get_tiling(self):
        a, b, p = C.c_int32(0), C.c_int32(0), C.c_int32(0)
        _check(lib().tbsma_get_tiling(self._h, C.byref(a), C.byref(b), C.byref(p)), "tbsma_get_tiling")
        return int(a.value), bool(b.value), bool(p.value)

    def describe_gather(self):
        n_tiles, box, persistent = self.get_tiling()
        if not n_tiles:
            return "thread per atom, records gathered through L1"
        how = ("persistent kernels (two CTAs of 16 warps per SM)" if persistent else
               "whole step in one cooperative kernel" if lib().tbsma_get_fused_step(self._h) == 1 else "one CTA per tile")
        return "%d %s tiles, %s" % (n_tiles, "box" if box else "layer", how)

    def set_tile(self, layers_per_tile, threads):
        _check(lib().tbsma_set_tile(self._h, int(layers_per_tile), int(threads)), "tbsma_set_tile")

    def set_graph(self, enable, conditional=True):
        _check(lib().tbsma_set_graph(self._h, (2 if conditional else 1) if enable else 0), "tbsma_set_graph")

    def set_outer_skin(self, outer_skin):
        _check(lib().tbsma_set_outer_skin(self._h, float(outer_skin)), "tbsma_set_outer_skin")

    def set_tile_split(self, ctas_per_tile):
        _check(lib().tbsma_set_tile_split(self._h, int(ctas_per_tile)), "tbsma_set_tile_split")

    def set_tile_box(self, force):
        _check(lib().tbsma_set_tile_box(self._h, int(bool(force))), "tbsma_set_tile_box")

    def set_fused_step(self, enable):
        _check(lib().tbsma_set_fused_step(self._h, int(bool(enable))), "tbsma_set_fused_step")

    def set_gather(self, mode):
        _check(lib().tbsma_set_gather(self._h, int(mode)), "tbsma_set_gather")

    def set_protocol(self, slab1_disp0=None, slab1_rate=None, stepwise_period=0, T_rate=None):
        """tbsma_set_protocol; device tensors (kept alive by the caller) or None; all None / 0 switches it off"""
        def ptr(t):
            return None if t is None else t.data_ptr()
        p = Protocol(ptr(slab1_disp0), ptr(slab1_rate), int(stepwise_period), ptr(T_rate))
        _check(lib().tbsma_set_protocol(self._h, C.byref(p)), "tbsma_set_protocol")

    def set_series(self, every=0, capacity=0, series=None, count=None, rupture_step=None, volume=None, L0=None):
        """tbsma_set_series; device tensors (kept alive by the caller); every = 0 switches recording off"""
        def ptr(t):
            return None if t is None else t.data_ptr()
        if not every:
            _check(lib().tbsma_set_series(self._h, None), "tbsma_set_series")
            return
        s = Series(int(every), int(capacity), ptr(series), ptr(count), ptr(rupture_step), ptr(volume), ptr(L0))
        _check(lib().tbsma_set_series(self._h, C.byref(s)), "tbsma_set_series")

    def series_histogram(self, series, count, capacity, col_x, col_y, x_lo, x_hi, nx, y_lo, y_hi, ny, hist, stream=None):
        _check(lib().tbsma_series_histogram(self._h, _dp(series), _dp(count), int(capacity), int(col_x), int(col_y),
                                            float(x_lo), float(x_hi), int(nx), float(y_lo), float(y_hi), int(ny),
                                            _dp(hist), _stream(stream)), "tbsma_series_histogram")

    def set_thermostat(self, kind, tau_fs=0.0):
        _check(lib().tbsma_set_thermostat(self._h, int(kind), float(tau_fs)), "tbsma_set_thermostat")

    def get_thermostat(self):
        xi, eta = np.zeros(self.R), np.zeros(self.R)
        _check(lib().tbsma_get_thermostat(self._h, _hp(xi), _hp(eta)), "tbsma_get_thermostat")
        return xi, eta

    def set_thermostat_state(self, xi, eta):
        xi = np.ascontiguousarray(xi, dtype=np.float64)
        eta = np.ascontiguousarray(eta, dtype=np.float64)
        assert len(xi) == self.R and len(eta) == self.R
        _check(lib().tbsma_set_thermostat_state(self._h, _hp(xi), _hp(eta)), "tbsma_set_thermostat_state")

    def set_stagger(self, enable):
        _check(lib().tbsma_set_stagger(self._h, int(bool(enable))), "tbsma_set_stagger")

    def set_balance(self, enable, cell=0.0):
        _check(lib().tbsma_set_balance(self._h, int(bool(enable)), float(cell)), "tbsma_set_balance")

    def set_async(self, enable, margin=0.03):
        _check(lib().tbsma_set_async(self._h, int(bool(enable)), float(margin)), "tbsma_set_async")

    def set_overlap(self, enable):
        _check(lib().tbsma_set_overlap(self._h, int(enable)), "tbsma_set_overlap")

    def set_timing(self, enable):
        _check(lib().tbsma_set_timing(self._h, int(bool(enable))), "tbsma_set_timing")

    def get_timing(self):
        """-> (dict of summed ms per kernel class, steps covered)"""
        ms = (C.c_double * 5)()
        n = C.c_int64(0)
        _check(lib().tbsma_get_timing(self._h, ms, C.byref(n)), "tbsma_get_timing")
        names = ("integrate", "rebuild", "density", "force", "finish")
        return {k: float(v) for k, v in zip(names, ms)}, int(n.value)

    def launch_count(self):
        return int(lib().tbsma_launch_count(self._h))


class DeviceState:
    """Device tensors of one workload (paper_1311_3890_b200.workloads.Workload) -- allocation only."""

    def __init__(self, w, device="cuda:0"):
        dev = torch.device(device)
        self.pos = torch.from_numpy(w.pos4.copy()).to(dev)
        self.vel = torch.from_numpy(w.vel4.copy()).to(dev)
        self.force = torch.zeros_like(self.pos)
        self.tag = torch.arange(w.n_atoms, dtype=torch.int32, device=dev)
        self.T = torch.from_numpy(np.ascontiguousarray(w.T, dtype=np.float32)).to(dev)
        self.seed = torch.from_numpy(np.ascontiguousarray(w.seed, dtype=np.uint64).view(np.int64).copy()).to(dev)
        self.slab_rate = torch.from_numpy(np.ascontiguousarray(w.slab_rate, dtype=np.float64)).to(dev)
        self.slab_disp = torch.zeros(w.n_replicas, dtype=torch.float64, device=dev)
        self.e_rep = torch.zeros(w.n_replicas, dtype=torch.float64, device=dev)
        self.w_rep = torch.zeros(w.n_replicas, 6, dtype=torch.float64, device=dev)
        self.ekin = torch.zeros(w.n_replicas, dtype=torch.float64, device=dev)

    def untag(self, t):
        """tensor in slot order -> numpy array in tag (original) order"""
        tag = self.tag.cpu().numpy()
        a = t.cpu().numpy()
        out = np.empty_like(a)
        out[tag] = a
        return out


def make_context(w, max_neighbors=112, params=None):
    """Context sized for a Workload."""
    ctx = Context(params, r_cut=w.r_cut, skin=w.skin)
    ctx.set_system(w.offsets, w.box_lo, w.box_hi, w.periodic, max_neighbors)
    return ctx
