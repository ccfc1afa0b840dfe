"""Thin ctypes binding of the C-ABI library (include/mcrt.h).  Argument marshalling only:
every step of the method runs in the CUDA kernels behind the `mcrt_*` calls.  PyTorch is used
for device buffers and streams.  There is no CPU fallback: a missing library or device raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

MCRT_HOST, MCRT_DEVICE = 0, 1
NOALLOC_MAX_SLOTS = 1 << 20          # MCRT_NOALLOC_MAX_SLOTS of include/mcrt.h
_lib = None


class McrtError(RuntimeError):
    pass


class _GridDesc(C.Structure):
    _fields_ = [("n_root", C.c_int32), ("sub", C.c_int32), ("origin", C.c_double * 3),
                ("root_size", C.c_double), ("refine", C.c_void_p), ("rho_root", C.c_void_p),
                ("rho_sub", C.c_void_p), ("mem", C.c_int), ("layout", C.c_int32)]


class _OpacityDesc(C.Structure):
    _fields_ = [("n_bins", C.c_int32), ("lambda_edges_um", C.c_void_p),
                ("n_species", C.c_int32), ("weight", C.c_void_p), ("kabs", C.c_void_p),
                ("ksca", C.c_void_p), ("g", C.c_void_p), ("T_min", C.c_double),
                ("T_max", C.c_double), ("n_T", C.c_int32)]


class _Source(C.Structure):
    _fields_ = [("type", C.c_int32), ("pos", C.c_double * 3), ("L", C.c_double),
                ("T_bb", C.c_double)]


class _ObserverDesc(C.Structure):
    _fields_ = [("n_mu", C.c_int32), ("n_pix", C.c_int32), ("dir", C.c_double * 3),
                ("half_angle_deg", C.c_double), ("half_width", C.c_double),
                ("bin_lo", C.c_int32), ("bin_hi", C.c_int32)]


class _Counters(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("emitted", "escaped", "lost", "absorptions",
                                          "scatterings", "flights", "crossings")]


class _PahDesc(C.Structure):
    _fields_ = [("n_C", C.c_int32), ("mass_fraction", C.c_double), ("kabs_pah", C.c_void_p),
                ("theta_K", C.c_double), ("T_lo", C.c_double), ("T_hi", C.c_double), ("n_Tp", C.c_int32)]


class _Results(C.Structure):
    _fields_ = [("n_abs", C.c_void_p), ("T", C.c_void_p), ("sed", C.c_void_p),
                ("emitted_per_bin", C.c_void_p), ("counters", C.POINTER(_Counters)),
                ("eps", C.POINTER(C.c_double))]


# every symbol include/mcrt.h declares (the stable boundary) ...
SYMBOLS_STABLE = ("mcrt_grid_create", "mcrt_destroy", "mcrt_leaf_slots", "mcrt_set_opacity",
                  "mcrt_set_source", "mcrt_run_batch", "mcrt_transport_batch",
                  "mcrt_update_temperature", "mcrt_store_slots", "mcrt_delta_words", "mcrt_transport_batch_delta",
                  "mcrt_accumulate_update", "mcrt_get_results", "mcrt_results_begin", "mcrt_results_wait",
                  "mcrt_get_cell_energy", "mcrt_get_cell_temperature", "mcrt_get_cell_temperature_noalloc",
                  "mcrt_get_sed", "mcrt_set_pah", "mcrt_get_pah_absorbed",
                  "mcrt_get_pah_emission_cdf", "mcrt_get_pah_temperature_distribution", "mcrt_set_observer",
                  "mcrt_get_sed_mu", "mcrt_get_image", "mcrt_get_counters", "mcrt_reset_tallies",
                  "mcrt_release_cached_memory", "mcrt_last_error")
# ... and include/mcrt_dev.h (tuning knobs, measurement tools, test hooks)
SYMBOLS_DEV = ("mcrt_gather_calibrate", "mcrt_set_launch", "mcrt_set_walk_quorum", "mcrt_set_tail_mode",
               "mcrt_set_source_order", "mcrt_set_cdf_guide", "mcrt_set_density_staging", "mcrt_density_staging",
               "mcrt_set_region_sweeps", "mcrt_get_region_sweep_counts", "mcrt_get_batch_times",
               "mcrt_get_tables", "mcrt_kernel_launches", "mcrt_debug_violations", "mcrt_philox_blocks",
               "mcrt_uniforms")
SYMBOLS = SYMBOLS_STABLE + SYMBOLS_DEV


def lib():
    """Load libmcrt.so (built in-tree by build.py).  Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        path = os.environ.get("MCRT_LIBRARY") or _build.LIB_PATH     # e.g. the -DMCRT_CHECKS variant
        if not os.path.exists(path):
            raise McrtError(f"{path} is missing: run `python -m paper_1201_3588_b200.build` "
                            "(there is no CPU fallback)")
        L = C.CDLL(path)
        vp, i32, i64, u64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64
        L.mcrt_grid_create.argtypes = [C.POINTER(_GridDesc), C.POINTER(vp)]
        L.mcrt_destroy.argtypes = [vp]
        L.mcrt_leaf_slots.restype = i64
        L.mcrt_leaf_slots.argtypes = [vp]
        L.mcrt_set_opacity.argtypes = [vp, C.POINTER(_OpacityDesc)]
        L.mcrt_set_source.argtypes = [vp, i32, C.POINTER(_Source)]
        L.mcrt_run_batch.argtypes = [vp, u64, u64, u64, vp]
        L.mcrt_transport_batch.argtypes = [vp, u64, u64, u64, vp]
        L.mcrt_update_temperature.argtypes = [vp, vp, u64, vp]
        L.mcrt_store_slots.restype = i64
        L.mcrt_store_slots.argtypes = [vp]
        L.mcrt_delta_words.restype = i64
        L.mcrt_delta_words.argtypes = [vp]
        L.mcrt_transport_batch_delta.argtypes = [vp, u64, u64, u64, vp, vp]
        L.mcrt_accumulate_update.argtypes = [vp, vp, u64, vp]
        L.mcrt_get_results.argtypes = [vp, C.POINTER(_Results), C.c_int]
        L.mcrt_results_begin.argtypes = [vp, C.POINTER(_Results), C.c_int, C.POINTER(i32)]
        L.mcrt_results_wait.argtypes = [vp, i32]
        L.mcrt_get_cell_energy.argtypes = [vp, vp, C.POINTER(C.c_double), C.c_int]
        L.mcrt_get_cell_temperature.argtypes = [vp, vp, C.c_int]
        L.mcrt_get_cell_temperature_noalloc.argtypes = [vp, vp]
        L.mcrt_get_cell_temperature_noalloc.restype = C.c_int
        L.mcrt_get_sed.argtypes = [vp, vp, C.c_int]
        L.mcrt_set_pah.argtypes = [vp, C.POINTER(_PahDesc)]
        L.mcrt_get_pah_absorbed.argtypes = [vp, vp, C.c_int]
        L.mcrt_get_pah_emission_cdf.argtypes = [vp, vp, C.c_int]
        L.mcrt_get_pah_temperature_distribution.argtypes = [vp, i64, vp, vp]
        L.mcrt_set_observer.argtypes = [vp, C.POINTER(_ObserverDesc)]
        L.mcrt_get_sed_mu.argtypes = [vp, vp, C.c_int]
        L.mcrt_get_image.argtypes = [vp, vp, C.c_int]
        L.mcrt_get_counters.argtypes = [vp, C.POINTER(_Counters), vp]
        L.mcrt_reset_tallies.argtypes = [vp, i32]
        L.mcrt_set_launch.argtypes = [vp, i32, i32]
        L.mcrt_set_walk_quorum.argtypes = [vp, i32]
        L.mcrt_set_tail_mode.argtypes = [vp, i32]
        L.mcrt_set_source_order.argtypes = [vp, i32]
        L.mcrt_set_cdf_guide.argtypes = [vp, i32]
        L.mcrt_set_cdf_guide.restype = C.c_int
        L.mcrt_set_region_sweeps.argtypes = [vp, i32, i32, i32, i32]
        L.mcrt_set_region_sweeps.restype = C.c_int
        L.mcrt_get_region_sweep_counts.argtypes = [vp, vp, i32, C.POINTER(i32)]
        L.mcrt_get_region_sweep_counts.restype = C.c_int
        L.mcrt_set_density_staging.argtypes = [vp, i32]
        L.mcrt_set_density_staging.restype = C.c_int
        L.mcrt_density_staging.argtypes = [vp]
        L.mcrt_density_staging.restype = i32
        L.mcrt_get_batch_times.argtypes = [vp, vp, vp, i32, C.POINTER(i32)]
        L.mcrt_get_tables.argtypes = [vp, vp, vp, vp]
        L.mcrt_kernel_launches.restype = i64
        L.mcrt_kernel_launches.argtypes = [vp]
        L.mcrt_debug_violations.restype = i64
        L.mcrt_debug_violations.argtypes = []
        L.mcrt_philox_blocks.argtypes = [vp, vp, vp, i64]
        L.mcrt_uniforms.argtypes = [vp, vp, vp, vp, i64]
        L.mcrt_gather_calibrate.argtypes = [u64, u64, C.POINTER(C.c_double), C.POINTER(C.c_double), vp]
        L.mcrt_gather_calibrate.restype = C.c_int
        L.mcrt_release_cached_memory.restype = i64
        L.mcrt_release_cached_memory.argtypes = []
        L.mcrt_last_error.restype = C.c_char_p
        L.mcrt_last_error.argtypes = [vp]
        for name in ("mcrt_grid_create", "mcrt_destroy", "mcrt_set_opacity", "mcrt_set_source",
                     "mcrt_run_batch", "mcrt_transport_batch", "mcrt_update_temperature",
                     "mcrt_transport_batch_delta", "mcrt_accumulate_update", "mcrt_get_results",
                     "mcrt_results_begin", "mcrt_results_wait", "mcrt_get_cell_energy", "mcrt_set_pah",
                     "mcrt_get_pah_absorbed", "mcrt_get_pah_emission_cdf",
                     "mcrt_get_pah_temperature_distribution", "mcrt_get_cell_temperature",
                     "mcrt_get_sed", "mcrt_set_observer", "mcrt_get_sed_mu", "mcrt_get_image",
                     "mcrt_get_counters", "mcrt_reset_tallies",
                     "mcrt_set_launch", "mcrt_set_walk_quorum", "mcrt_set_tail_mode", "mcrt_set_source_order",
                     "mcrt_get_batch_times",
                     "mcrt_get_tables",
                     "mcrt_philox_blocks", "mcrt_uniforms"):
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _np_ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _is_tensor(x):
    return hasattr(x, "data_ptr")


class Context:
    """mcrt_ctx with the call names of include/mcrt.h.  Inputs may be numpy arrays (host) or
    torch CUDA tensors (device); outputs are numpy arrays, or torch CUDA tensors with
    device=True."""

    def __init__(self):
        self.h = None
        self.n_bins = 0
        self.n_T = 0
        self._keep = None

    # -- errors ---------------------------------------------------------------------------
    def _check(self, rc, what):
        if rc != 0:
            msg = lib().mcrt_last_error(self.h)
            raise McrtError(f"{what}: status {rc}: {msg.decode() if msg else ''}")

    # -- set-up ---------------------------------------------------------------------------
    def grid_create(self, n_root, sub, origin, root_size, refine, rho_root, rho_sub, layout=0):
        L = lib()
        d = _GridDesc()
        d.n_root, d.sub = int(n_root), int(sub)
        d.layout = int(layout)
        d.origin = (C.c_double * 3)(*[float(v) for v in origin])
        d.root_size = float(root_size)
        if _is_tensor(rho_root):
            import torch
            keep = [rho_root.contiguous().to(torch.float32)]
            d.rho_root = keep[0].data_ptr()
            if refine is not None:
                keep.append(refine.contiguous().to(torch.uint8))
                d.refine = keep[-1].data_ptr()
            if rho_sub is not None:
                keep.append(rho_sub.contiguous().to(torch.float32))
                d.rho_sub = keep[-1].data_ptr()
            d.mem = MCRT_DEVICE
        else:
            keep = [np.ascontiguousarray(rho_root, dtype=np.float32)]
            d.rho_root = _np_ptr(keep[0])
            if refine is not None:
                keep.append(np.ascontiguousarray(refine, dtype=np.uint8))
                d.refine = _np_ptr(keep[-1])
            if rho_sub is not None:
                keep.append(np.ascontiguousarray(rho_sub, dtype=np.float32))
                d.rho_sub = _np_ptr(keep[-1])
            d.mem = MCRT_HOST
        out = C.c_void_p()
        rc = L.mcrt_grid_create(C.byref(d), C.byref(out))
        if rc != 0:
            msg = L.mcrt_last_error(None)
            raise McrtError(f"mcrt_grid_create: status {rc}: {msg.decode() if msg else ''}")
        self.h = out
        self.slots = int(L.mcrt_leaf_slots(self.h))
        return self

    def set_opacity(self, lambda_edges_um, weight, kabs, ksca, g, T_min=0.0, T_max=0.0, n_T=0):
        e = np.ascontiguousarray(lambda_edges_um, dtype=np.float64)
        w = np.ascontiguousarray(weight, dtype=np.float64)
        ka = np.ascontiguousarray(kabs, dtype=np.float32).reshape(len(w), -1)
        ks = np.ascontiguousarray(ksca, dtype=np.float32).reshape(len(w), -1)
        gg = np.ascontiguousarray(g, dtype=np.float32).reshape(len(w), -1)
        d = _OpacityDesc()
        d.n_bins, d.n_species = len(e) - 1, len(w)
        d.lambda_edges_um, d.weight = _np_ptr(e), _np_ptr(w)
        d.kabs, d.ksca, d.g = _np_ptr(ka), _np_ptr(ks), _np_ptr(gg)
        d.T_min, d.T_max, d.n_T = float(T_min), float(T_max), int(n_T)
        self._check(lib().mcrt_set_opacity(self.h, C.byref(d)), "mcrt_set_opacity")
        self.n_bins = d.n_bins
        self.n_T = n_T if n_T > 0 else 801
        return self

    def set_pah(self, n_C, mass_fraction, kabs_pah, theta_K=500.0, T_lo=5.0, T_hi=1.0e4, n_Tp=128):
        """Declare the transiently heated PAH (after set_opacity)."""
        k = np.ascontiguousarray(kabs_pah, dtype=np.float32)
        d = _PahDesc()
        d.n_C, d.mass_fraction, d.kabs_pah = int(n_C), float(mass_fraction), _np_ptr(k)
        d.theta_K, d.T_lo, d.T_hi, d.n_Tp = float(theta_K), float(T_lo), float(T_hi), int(n_Tp)
        self._check(lib().mcrt_set_pah(self.h, C.byref(d)), "mcrt_set_pah")
        self.n_Tp = int(n_Tp) if n_Tp else 128
        return self

    def get_pah_absorbed(self, device=False):
        out, p, mem = self._out((self.slots, self.n_bins), np.uint32, device)
        self._check(lib().mcrt_get_pah_absorbed(self.h, p, mem), "mcrt_get_pah_absorbed")
        return out

    def get_pah_emission_cdf(self, device=False):
        out, p, mem = self._out((self.slots, self.n_bins), np.float32, device)
        self._check(lib().mcrt_get_pah_emission_cdf(self.h, p, mem), "mcrt_get_pah_emission_cdf")
        return out

    def get_pah_temperature_distribution(self, leaf_slot):
        T, P = np.zeros(self.n_Tp), np.zeros(self.n_Tp)
        self._check(lib().mcrt_get_pah_temperature_distribution(self.h, int(leaf_slot), _np_ptr(T), _np_ptr(P)),
                    "mcrt_get_pah_temperature_distribution")
        return T, P

    def set_source(self, sources):
        arr = (_Source * len(sources))()
        for i, s in enumerate(sources):
            arr[i].type = int(s.type)
            arr[i].pos = (C.c_double * 3)(*[float(v) for v in s.pos])
            arr[i].L, arr[i].T_bb = float(s.L), float(s.T_bb)
        self._check(lib().mcrt_set_source(self.h, len(sources), arr), "mcrt_set_source")
        return self

    # -- hot path -------------------------------------------------------------------------
    def run_batch(self, seed, first_packet_id, n_packets, stream=None):
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        self._check(lib().mcrt_run_batch(self.h, int(seed), int(first_packet_id),
                                         int(n_packets), C.c_void_p(stream)), "mcrt_run_batch")

    def transport_batch(self, seed, first_packet_id, n_packets, stream=None):
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        self._check(lib().mcrt_transport_batch(self.h, int(seed), int(first_packet_id),
                                               int(n_packets), C.c_void_p(stream)),
                    "mcrt_transport_batch")

    def update_temperature(self, tally_sum=None, n_cum=0, stream=None):
        """tally_sum: torch int64 CUDA tensor [leaf slots] (sum over ranks) or None."""
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        p = None if tally_sum is None else C.c_void_p(tally_sum.data_ptr())
        self._check(lib().mcrt_update_temperature(self.h, p, int(n_cum), C.c_void_p(stream)),
                    "mcrt_update_temperature")

    def transport_batch_delta(self, seed, first_packet_id, n_packets, stream=None):
        """This rank's share of a batch, tallied into a per-batch uint32 array in the library's
        storage order (a torch int32 CUDA tensor owned by this object, reused every batch): the
        array the ranks of a packet-sharded run all-reduce."""
        import torch
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        words = int(lib().mcrt_delta_words(self.h))                # (grows when a PAH is declared)
        if getattr(self, "_delta", None) is None or self._delta.numel() != words:
            self._delta = torch.empty(words, dtype=torch.int32, device="cuda")
        self._check(lib().mcrt_transport_batch_delta(self.h, int(seed), int(first_packet_id), int(n_packets),
                                                     C.c_void_p(self._delta.data_ptr()), C.c_void_p(stream)),
                    "mcrt_transport_batch_delta")
        return self._delta

    def accumulate_update(self, delta_sum, n_cum, stream=None):
        """Adds the batch's counts summed over ranks to the cumulative tally and updates T."""
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        self._check(lib().mcrt_accumulate_update(self.h, C.c_void_p(delta_sum.data_ptr()), int(n_cum),
                                                 C.c_void_p(stream)), "mcrt_accumulate_update")

    # -- results --------------------------------------------------------------------------
    def _results_struct(self, bufs):
        """bufs: dict with any of n_abs / T / sed / emitted_per_bin -> numpy arrays (host, ideally
        views of pinned memory) or torch CUDA tensors; returns (struct, keep-alive, mem)."""
        r = _Results()
        dev = any(_is_tensor(v) for v in bufs.values())
        for k in ("n_abs", "T", "sed", "emitted_per_bin"):
            v = bufs.get(k)
            if v is not None:
                setattr(r, k, v.data_ptr() if _is_tensor(v) else v.ctypes.data)
        c, eps = _Counters(), C.c_double(0)
        r.counters, r.eps = C.pointer(c), C.pointer(eps)
        return r, (c, eps, bufs), MCRT_DEVICE if dev else MCRT_HOST

    def results_begin(self, bufs):
        """Queue the read-out of a finished batch into `bufs` (see _results_struct); the next
        run_batch may be issued at once.  Returns a handle for results_wait."""
        r, keep, mem = self._results_struct(bufs)
        t = C.c_int32(-1)
        self._check(lib().mcrt_results_begin(self.h, C.byref(r), mem, C.byref(t)), "mcrt_results_begin")
        return (t.value, r, keep)

    def results_wait(self, handle):
        t, r, (c, eps, bufs) = handle
        self._check(lib().mcrt_results_wait(self.h, t), "mcrt_results_wait")
        out = dict(bufs)
        out["counters"] = {n: int(getattr(c, n)) for n, _ in _Counters._fields_}
        out["eps"] = eps.value
        return out

    def get_results(self, bufs):
        """Everything in one call and one synchronisation."""
        return self.results_wait(self.results_begin(bufs))

    def _out(self, shape, np_dtype, device, out=None):
        """Output buffer: a torch CUDA tensor (device=True), the caller's `out` (a C-contiguous
        numpy array of the right shape and dtype -- e.g. a view of pinned memory, reused from
        call to call), or a fresh numpy array."""
        if device:
            import torch
            t = torch.empty(shape, dtype=getattr(torch, np.dtype(np_dtype).name
                                                 .replace("uint64", "int64").replace("uint32", "int32")),
                            device="cuda")
            return t, C.c_void_p(t.data_ptr()), MCRT_DEVICE
        if out is not None:
            if out.shape != tuple(shape) or out.dtype != np.dtype(np_dtype) or not out.flags.c_contiguous:
                raise McrtError(f"out must be a C-contiguous {np.dtype(np_dtype)} array of shape {tuple(shape)}")
            return out, _np_ptr(out), MCRT_HOST
        a = np.zeros(shape, dtype=np_dtype)
        return a, _np_ptr(a), MCRT_HOST

    def get_cell_energy(self, device=False, out=None):
        out, p, mem = self._out((self.slots,), np.uint64, device, out)
        eps = C.c_double(0)
        self._check(lib().mcrt_get_cell_energy(self.h, p, C.byref(eps), mem),
                    "mcrt_get_cell_energy")
        return out, eps.value

    def get_cell_temperature(self, device=False, out=None):
        out, p, mem = self._out((self.slots,), np.float32, device, out)
        self._check(lib().mcrt_get_cell_temperature(self.h, p, mem),
                    "mcrt_get_cell_temperature")
        return out

    def get_cell_temperature_noalloc(self, out=None):
        """Temperatures [leaf slots] in K as a numpy array, read out without any device allocation
        by the library (mcrt_get_cell_temperature_noalloc): for callers that cannot cudaMalloc
        between batches -- all device memory already owned by another pool or a fixed quota,
        another thread recording a CUDA graph, a loop that cannot take an allocation's stall.
        Grids of up to NOALLOC_MAX_SLOTS leaf slots; larger ones raise McrtError.  Same values
        bit for bit as get_cell_temperature().  One library-owned array per GPU serves all
        calls, so the library runs them one at a time."""
        out, p, _ = self._out((self.slots,), np.float32, False, out)
        self._check(lib().mcrt_get_cell_temperature_noalloc(self.h, p),
                    "mcrt_get_cell_temperature_noalloc")
        return out

    def get_sed(self, device=False, out=None):
        out, p, mem = self._out((3, self.n_bins), np.uint64, device, out)
        self._check(lib().mcrt_get_sed(self.h, p, mem), "mcrt_get_sed")
        return out

    def set_observer(self, n_mu=0, n_pix=0, direction=(0.0, 0.0, 1.0), half_angle_deg=5.0,
                     half_width_cm=1.0, bin_lo=0, bin_hi=-1):
        d = _ObserverDesc()
        d.n_mu, d.n_pix = int(n_mu), int(n_pix)
        d.dir = (C.c_double * 3)(*[float(v) for v in direction])
        d.half_angle_deg, d.half_width = float(half_angle_deg), float(half_width_cm)
        d.bin_lo, d.bin_hi = int(bin_lo), int(bin_hi)
        self._check(lib().mcrt_set_observer(self.h, C.byref(d)), "mcrt_set_observer")
        self.n_mu, self.n_pix = d.n_mu, d.n_pix

    def get_sed_mu(self, device=False):
        out, p, mem = self._out((self.n_mu, 3, self.n_bins), np.uint64, device)
        self._check(lib().mcrt_get_sed_mu(self.h, p, mem), "mcrt_get_sed_mu")
        return out

    def get_image(self, device=False):
        out, p, mem = self._out((self.n_pix, self.n_pix), np.uint64, device)
        self._check(lib().mcrt_get_image(self.h, p, mem), "mcrt_get_image")
        return out

    def get_counters(self, out=None):
        c = _Counters()
        e = np.zeros(self.n_bins, dtype=np.uint64) if out is None else out
        self._check(lib().mcrt_get_counters(self.h, C.byref(c), _np_ptr(e)),
                    "mcrt_get_counters")
        d = {n: int(getattr(c, n)) for n, _ in _Counters._fields_}
        d["emitted_per_bin"] = e
        return d

    def reset_tallies(self, what=3):
        self._check(lib().mcrt_reset_tallies(self.h, int(what)), "mcrt_reset_tallies")

    # -- tuning / introspection ---------------------------------------------------------
    def set_launch(self, threads_per_block=0, blocks_per_sm=0):
        self._check(lib().mcrt_set_launch(self.h, threads_per_block, blocks_per_sm),
                    "mcrt_set_launch")

    def set_walk_quorum(self, quorum):
        self._check(lib().mcrt_set_walk_quorum(self.h, int(quorum)), "mcrt_set_walk_quorum")

    def set_tail_mode(self, mode):
        self._check(lib().mcrt_set_tail_mode(self.h, int(mode)), "mcrt_set_tail_mode")

    def set_region_sweeps(self, sweeps, shape=(0, 0, 0)):
        self._check(lib().mcrt_set_region_sweeps(self.h, int(sweeps), *[int(v) for v in shape]),
                    "mcrt_set_region_sweeps")

    def get_region_sweep_counts(self):
        out = np.zeros(32, dtype=np.uint32)
        n = C.c_int32(0)
        self._check(lib().mcrt_get_region_sweep_counts(self.h, _np_ptr(out), 32, C.byref(n)),
                    "mcrt_get_region_sweep_counts")
        return out[:n.value].copy()

    def set_density_staging(self, mode):
        self._check(lib().mcrt_set_density_staging(self.h, int(mode)), "mcrt_set_density_staging")

    def density_staging(self):
        return int(lib().mcrt_density_staging(self.h))

    def set_cdf_guide(self, on=True):
        self._check(lib().mcrt_set_cdf_guide(self.h, 1 if on else 0), "mcrt_set_cdf_guide")

    def set_source_order(self, mode):
        self._check(lib().mcrt_set_source_order(self.h, int(mode)), "mcrt_set_source_order")

    def get_batch_times(self, cap=4096):
        t = np.zeros(cap, dtype=np.float32)
        u = np.zeros(cap, dtype=np.float32)
        n = C.c_int32(0)
        self._check(lib().mcrt_get_batch_times(self.h, _np_ptr(t), _np_ptr(u), cap,
                                               C.byref(n)), "mcrt_get_batch_times")
        return t[:n.value].copy(), u[:n.value].copy()

    def get_tables(self):
        opac = np.zeros((self.n_bins, 4), dtype=np.float32)
        lnQ = np.zeros(self.n_T, dtype=np.float32)
        cdf = np.zeros((self.n_T, self.n_bins), dtype=np.float32)
        self._check(lib().mcrt_get_tables(self.h, _np_ptr(opac), _np_ptr(lnQ), _np_ptr(cdf)),
                    "mcrt_get_tables")
        return opac, lnQ, cdf

    def store_slots(self):
        """Length of the library's internal storage of the leaf arrays (>= slots: bricks are padded)."""
        return int(lib().mcrt_store_slots(self.h))

    def kernel_launches(self):
        return int(lib().mcrt_kernel_launches(self.h))

    def destroy(self):
        if self.h is not None and _lib is not None:
            _lib.mcrt_destroy(self.h)
        self.h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def from_workload(wl, device_inputs=False, n_T=0, T_min=0.0, T_max=0.0, layout=0) -> Context:
    """grid_create -> set_opacity -> set_source for a workloads.Workload."""
    ctx = Context()
    refine, rho_root, rho_sub = wl.refine, wl.rho_root, wl.rho_sub
    if device_inputs:
        import torch
        rho_root = torch.from_numpy(np.ascontiguousarray(rho_root)).cuda()
        refine = None if refine is None else torch.from_numpy(np.ascontiguousarray(refine)).cuda()
        rho_sub = None if rho_sub is None else torch.from_numpy(np.ascontiguousarray(rho_sub)).cuda()
    ctx.grid_create(wl.n_root, wl.sub, wl.origin, wl.root_size, refine, rho_root, rho_sub,
                    layout)
    ctx.set_opacity(wl.lambda_edges_um, wl.weight, wl.kabs, wl.ksca, wl.g, T_min, T_max, n_T)
    ctx.set_source(wl.sources)
    return ctx


def run_workload(wl, n_packets=None, batch=None, **kw) -> Context:
    ctx = from_workload(wl, **kw)
    for first, cnt in wl.batches(n_packets, batch):
        ctx.run_batch(wl.seed, first, cnt)
    return ctx


def philox_blocks(key2, ctr):
    k = np.ascontiguousarray(key2, dtype=np.uint32)
    c = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    o = np.zeros_like(c)
    rc = lib().mcrt_philox_blocks(_np_ptr(k), _np_ptr(c), _np_ptr(o), len(c))
    if rc != 0:
        raise McrtError(f"mcrt_philox_blocks: status {rc}: {lib().mcrt_last_error(None).decode()}")
    return o


def uniforms(words):
    """(fp32 uniform, fp64 uniform, -ln of the fp32 uniform) the kernels derive from random words."""
    w = np.ascontiguousarray(words, dtype=np.uint32).ravel()
    u = np.zeros(len(w), dtype=np.float32)
    ud = np.zeros(len(w), dtype=np.float64)
    tau = np.zeros(len(w), dtype=np.float32)
    rc = lib().mcrt_uniforms(_np_ptr(w), _np_ptr(u), _np_ptr(ud), _np_ptr(tau), len(w))
    if rc != 0:
        raise McrtError(f"mcrt_uniforms: status {rc}: {lib().mcrt_last_error(None).decode()}")
    return u, ud, tau


def gather_calibrate(footprint_bytes, n_gathers=1 << 30, stream=None):
    """Independent 4-byte gathers per second over an array of `footprint_bytes` (gather roofline)."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    g, sec = C.c_double(0), C.c_double(0)
    rc = lib().mcrt_gather_calibrate(int(footprint_bytes), int(n_gathers), C.byref(g), C.byref(sec),
                                     C.c_void_p(stream))
    if rc != 0:
        raise McrtError(f"mcrt_gather_calibrate: status {rc}: {lib().mcrt_last_error(None).decode()}")
    return g.value, sec.value


def release_cached_memory():
    """Give the device blocks the library caches after contexts were destroyed back to the driver;
    returns the bytes released."""
    return int(lib().mcrt_release_cached_memory())


def debug_violations():
    """Out-of-range storage indices seen by a -DMCRT_CHECKS library (-1: built without checks)."""
    return int(lib().mcrt_debug_violations())
