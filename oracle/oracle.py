"""ctypes front end of the fp64 CPU oracle (oracle/mcrt_oracle.cpp).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference leg may import this.  It never touches the CUDA path and shares no code
with it (the seeded input generators in paper_1201_3588_b200/workloads.py are the only
common module, and they hold none of the method's arithmetic).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mcrt_oracle.cpp")
_LIB = os.path.join(_HERE, "libmcrt_oracle.so")
_lib = None


_LIB_SAN = os.path.join(_HERE, "libmcrt_oracle_san.so")


def build(force: bool = False, sanitize: bool = False) -> str:
    """Compile the oracle with g++ (-O2, OpenMP).  Building the checker is not using it.
    sanitize=True builds a second library with -fsanitize=address,undefined (SURVEY.md
    section 5); tests/test_oracle_sanitizers.py runs the pins' workloads on it in a
    subprocess (LD_PRELOAD of libasan, MCRT_ORACLE_LIBRARY pointing at it)."""
    out = _LIB_SAN if sanitize else _LIB
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
        tmp = out + ".tmp.%d" % os.getpid()
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                 "-fno-omit-frame-pointer"] if sanitize else ["-O2"]
        subprocess.check_call(["g++"] + flags + ["-std=c++17", "-fopenmp", "-shared", "-fPIC",
                               "-o", tmp, _SRC])
        os.replace(tmp, out)
    return out


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(os.environ.get("MCRT_ORACLE_LIBRARY") or build())
        L = _lib
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_double, C.c_void_p,
                                 C.c_void_p, C.c_void_p]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_leaf_slots.restype = C.c_int64
        L.orc_leaf_slots.argtypes = [C.c_void_p]
        L.orc_set_walker.argtypes = [C.c_void_p, C.c_int]
        L.orc_set_opacity.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p,
                                      C.c_void_p, C.c_void_p, C.c_void_p, C.c_double,
                                      C.c_double, C.c_int]
        L.orc_set_source.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p]
        L.orc_run_batch.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64, C.c_int]
        L.orc_transport_batch.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64,
                                          C.c_int]
        L.orc_update_temperature.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
        L.orc_set_observer.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_double,
                                       C.c_double, C.c_int, C.c_int]
        L.orc_get_observer_axes.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_get_sed_mu.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_get_image.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_run_bw.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint64]
        L.orc_trace_packet.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_int, C.c_void_p,
                                       C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_get_cell_energy.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_get_cell_temperature.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_set_cell_temperature.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_get_sed.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_get_counters.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_reset_tallies.argtypes = [C.c_void_p, C.c_int]
        L.orc_get_tables.argtypes = [C.c_void_p] + [C.c_void_p] * 8
        L.orc_get_source_cdf.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_philox.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_draw4.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p]
        L.orc_isotropic.argtypes = [C.c_double, C.c_double, C.c_void_p]
        L.orc_hg_cos.restype = C.c_double
        L.orc_hg_cos.argtypes = [C.c_double, C.c_double]
        L.orc_rotate.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_void_p]
        L.orc_planck.restype = C.c_double
        L.orc_planck.argtypes = [C.c_double, C.c_double]
        L.orc_sample_emission_bin.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
        L.orc_temperature_from_q.restype = C.c_double
        L.orc_temperature_from_q.argtypes = [C.c_void_p, C.c_double]
        L.orc_leaf_mass.restype = C.c_double
        L.orc_leaf_mass.argtypes = [C.c_void_p, C.c_int64]
        L.orc_emit.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64] + [C.c_void_p] * 4
        L.orc_walk.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int,
                               C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_set_pah.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_void_p, C.c_double,
                                  C.c_double, C.c_int]
        L.orc_get_pah_grid.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        L.orc_pah_solve.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_pah_rates.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_uint64, C.c_void_p]
        L.orc_pah_update.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
        L.orc_pah_enthalpy.restype = C.c_double
        L.orc_pah_enthalpy.argtypes = [C.c_void_p, C.c_double]
        L.orc_pah_heat_capacity.restype = C.c_double
        L.orc_pah_heat_capacity.argtypes = [C.c_void_p, C.c_double]
        L.orc_get_pah_absorbed.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_get_pah_cdf.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_max_threads.restype = C.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


COUNTER_NAMES = ("emitted", "escaped", "lost", "absorptions", "scatterings", "flights",
                 "crossings")


class Oracle:
    """Same call sequence as the C-ABI: grid -> opacity -> source -> run_batch -> getters."""

    def __init__(self, wl, n_T: int = 0, T_min: float = 0.0, T_max: float = 0.0):
        L = lib()
        origin = np.asarray(wl.origin, dtype=np.float64)
        refine = None if wl.refine is None else np.ascontiguousarray(wl.refine, dtype=np.uint8)
        rho_root = np.ascontiguousarray(wl.rho_root, dtype=np.float32)
        rho_sub = None if wl.rho_sub is None else np.ascontiguousarray(wl.rho_sub, np.float32)
        self.h = L.orc_create(wl.n_root, wl.sub, _p(origin), float(wl.root_size), _p(refine),
                              _p(rho_root), _p(rho_sub))
        if not self.h:
            raise ValueError("orc_create failed")
        self.wl = wl
        self.nb = wl.n_bins
        self.slots = int(L.orc_leaf_slots(self.h))
        edges = np.ascontiguousarray(wl.lambda_edges_um, dtype=np.float64)
        w = np.ascontiguousarray(wl.weight, dtype=np.float64)
        ka = np.ascontiguousarray(wl.kabs, dtype=np.float32)
        ks = np.ascontiguousarray(wl.ksca, dtype=np.float32)
        g = np.ascontiguousarray(wl.g, dtype=np.float32)
        rc = L.orc_set_opacity(self.h, self.nb, _p(edges), len(w), _p(w), _p(ka), _p(ks),
                               _p(g), T_min, T_max, n_T)
        assert rc == 0
        self.n_T = n_T if n_T > 0 else 801
        ty = np.array([s.type for s in wl.sources], dtype=np.int32)
        pos = np.array([s.pos for s in wl.sources], dtype=np.float64).reshape(-1)
        Ls = np.array([s.L for s in wl.sources], dtype=np.float64)
        Tb = np.array([s.T_bb for s in wl.sources], dtype=np.float64)
        rc = L.orc_set_source(self.h, len(ty), _p(ty), _p(pos), _p(Ls), _p(Tb))
        assert rc == 0
        self.n_src = len(ty)

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_destroy(self.h)
            self.h = None

    # ---- O11..O13: transiently heated PAH ----
    def set_pah(self, n_C, mass_fraction, kabs_pah, theta_K=500.0, T_lo=5.0, T_hi=1.0e4, n_Tp=128):
        k = np.ascontiguousarray(kabs_pah, dtype=np.float32)
        assert k.shape == (self.nb,)
        rc = lib().orc_set_pah(self.h, int(n_C), float(mass_fraction), float(theta_K), _p(k), float(T_lo),
                               float(T_hi), int(n_Tp))
        assert rc == 0
        self.n_Tp = int(n_Tp)

    def pah_grid(self):
        T, U, Lam = np.zeros(self.n_Tp), np.zeros(self.n_Tp), np.zeros(self.n_Tp)
        Cmol, q = np.zeros(self.nb), np.zeros(self.nb)
        lib().orc_get_pah_grid(self.h, _p(T), _p(U), _p(Lam), _p(Cmol), _p(q))
        return dict(T=T, U=U, Lam=Lam, Cmol=Cmol, q=q)

    def pah_solve(self, R):
        R = np.ascontiguousarray(R, dtype=np.float64)
        P, cdf = np.zeros(self.n_Tp), np.zeros(self.nb)
        lib().orc_pah_solve(self.h, _p(R), _p(P), _p(cdf))
        return P, cdf

    def pah_rates(self, slot, counts, n_cum):
        c = np.ascontiguousarray(counts, dtype=np.uint64)
        R = np.zeros(self.nb)
        ok = lib().orc_pah_rates(self.h, int(slot), _p(c), int(n_cum), _p(R))
        return R if ok else None

    def pah_update(self, counts, n_cum):
        c = np.ascontiguousarray(counts, dtype=np.uint64)
        assert c.size == self.slots * self.nb
        lib().orc_pah_update(self.h, _p(c), int(n_cum))

    def pah_enthalpy(self, T):
        return lib().orc_pah_enthalpy(self.h, float(T))

    def pah_heat_capacity(self, T):
        return lib().orc_pah_heat_capacity(self.h, float(T))

    def pah_absorbed(self):
        out = np.zeros((self.slots, self.nb), dtype=np.uint64)
        tot = C.c_uint64(0)
        lib().orc_get_pah_absorbed(self.h, _p(out), C.byref(tot))
        return out, tot.value

    def pah_cdf(self):
        out = np.zeros((self.slots, self.nb))
        lib().orc_get_pah_cdf(self.h, _p(out))
        return out

    def set_walker(self, w: int):
        lib().orc_set_walker(self.h, w)

    def run_batch(self, seed: int, first: int, n: int, threads: int = 0):
        rc = lib().orc_run_batch(self.h, seed, first, n, threads)
        assert rc == 0

    def transport_batch(self, seed: int, first: int, n: int, threads: int = 0):
        """Transport only (T frozen, no temperature update): one rank's share of a batch."""
        rc = lib().orc_transport_batch(self.h, seed, first, n, threads)
        assert rc == 0

    def update_temperature(self, tally_sum, n_cum: int):
        """O7 on counts summed over ranks."""
        t = np.ascontiguousarray(tally_sum, dtype=np.uint64)
        assert t.shape == (self.slots,)
        rc = lib().orc_update_temperature(self.h, _p(t), int(n_cum))
        assert rc == 0

    def run_bw(self, seed: int, first: int, n: int, n_total: int):
        """O10: the original serial scheme (immediate T update + Bjorkman-Wood correction)."""
        rc = lib().orc_run_bw(self.h, seed, first, n, n_total)
        assert rc == 0

    def run(self, n_packets=None, batch=None, threads: int = 0):
        for first, cnt in self.wl.batches(n_packets, batch):
            self.run_batch(self.wl.seed, first, cnt, threads)
        return self

    def cell_energy(self):
        n = np.zeros(self.slots, dtype=np.uint64)
        eps = C.c_double(0)
        lib().orc_get_cell_energy(self.h, _p(n), C.byref(eps))
        return n, eps.value

    def cell_temperature(self):
        T = np.zeros(self.slots, dtype=np.float64)
        lib().orc_get_cell_temperature(self.h, _p(T))
        return T

    def set_cell_temperature(self, T):
        T = np.ascontiguousarray(np.broadcast_to(np.asarray(T, np.float64), (self.slots,)))
        lib().orc_set_cell_temperature(self.h, _p(T))

    def set_observer(self, n_mu=0, n_pix=0, direction=(0.0, 0.0, 1.0), half_angle_deg=5.0,
                     half_width_cm=1.0, bin_lo=0, bin_hi=-1):
        """O9 (R34): inclination-binned SED and escape-direction image."""
        d = np.ascontiguousarray(direction, dtype=np.float64)
        if bin_hi < 0:
            bin_hi = self.nb - 1
        rc = lib().orc_set_observer(self.h, n_mu, n_pix, _p(d), float(half_angle_deg),
                                    float(half_width_cm), int(bin_lo), int(bin_hi))
        assert rc == 0
        self.n_mu, self.n_pix = n_mu, n_pix

    def observer_axes(self):
        o, e1, e2 = np.zeros(3), np.zeros(3), np.zeros(3)
        lib().orc_get_observer_axes(self.h, _p(o), _p(e1), _p(e2))
        return o, e1, e2

    def sed_mu(self):
        s = np.zeros((self.n_mu, 3, self.nb), dtype=np.uint64)
        lib().orc_get_sed_mu(self.h, _p(s))
        return s

    def image(self):
        s = np.zeros((self.n_pix, self.n_pix), dtype=np.uint64)
        lib().orc_get_image(self.h, _p(s))
        return s

    def sed(self):
        s = np.zeros((3, self.nb), dtype=np.uint64)
        lib().orc_get_sed(self.h, _p(s))
        return s

    def counters(self):
        c = np.zeros(7, dtype=np.uint64)
        e = np.zeros(self.nb, dtype=np.uint64)
        lib().orc_get_counters(self.h, _p(c), _p(e))
        d = {k: int(v) for k, v in zip(COUNTER_NAMES, c)}
        d["emitted_per_bin"] = e
        return d

    def reset_tallies(self, what: int = 3):
        lib().orc_reset_tallies(self.h, what)

    def tables(self):
        nb, nT = self.nb, self.n_T
        out = {k: np.zeros(nb) for k in ("nu", "dnu", "kabs", "kext", "alb", "g")}
        out["Q"] = np.zeros(nT)
        out["C"] = np.zeros((nT, nb))
        lib().orc_get_tables(self.h, *[_p(out[k]) for k in
                                       ("nu", "dnu", "kabs", "kext", "alb", "g", "Q", "C")])
        cs = np.zeros((self.n_src, nb))
        lc = np.zeros(self.n_src)
        lib().orc_get_source_cdf(self.h, _p(cs), _p(lc))
        out["Csrc"], out["Lcdf"] = cs, lc
        return out

    def trace_packet(self, seed: int, pid: int, cap: int = 4096):
        ty = np.zeros(cap, dtype=np.int32)
        bn = np.zeros(cap, dtype=np.int32)
        sl = np.zeros(cap, dtype=np.int64)
        xyz = np.zeros((cap, 3), dtype=np.float64)
        n = lib().orc_trace_packet(self.h, seed, pid, cap, _p(ty), _p(bn), _p(sl), _p(xyz))
        return ty[:n], bn[:n], sl[:n], xyz[:n]

    def emit(self, seed: int, pid: int):
        x = np.zeros(3)
        d = np.zeros(3)
        b = C.c_int(0)
        s = C.c_int64(0)
        lib().orc_emit(self.h, seed, pid, _p(x), _p(d), C.byref(b), C.byref(s))
        return x, d, b.value, s.value

    def walk(self, x, d, bin_, tau_star, walker=0):
        x = np.ascontiguousarray(x, dtype=np.float64)
        d = np.ascontiguousarray(d, dtype=np.float64)
        xo = np.zeros(3)
        slot = C.c_int64(-1)
        cr = C.c_uint64(0)
        r = lib().orc_walk(self.h, walker, _p(x), _p(d), bin_, tau_star, C.byref(slot), _p(xo),
                           C.byref(cr))
        return r, slot.value, xo, cr.value

    def sample_emission_bin(self, T, u0, u1):
        return lib().orc_sample_emission_bin(self.h, T, u0, u1)

    def temperature_from_q(self, q):
        return lib().orc_temperature_from_q(self.h, q)

    def leaf_mass(self, slot):
        return lib().orc_leaf_mass(self.h, slot)


# component functions ---------------------------------------------------------------------
def philox(key, ctr):
    k = np.asarray(key, dtype=np.uint32)
    c = np.asarray(ctr, dtype=np.uint32)
    o = np.zeros(4, dtype=np.uint32)
    lib().orc_philox(_p(k), _p(c), _p(o))
    return o


def draw4(seed, pid, k, tag):
    u = np.zeros(4)
    lib().orc_draw4(seed, pid, k, tag, _p(u))
    return u


def isotropic(u2, u3):
    d = np.zeros(3)
    lib().orc_isotropic(u2, u3, _p(d))
    return d


def hg_cos(g, u):
    return lib().orc_hg_cos(g, u)


def rotate(d, ct, phi):
    d = np.ascontiguousarray(d, dtype=np.float64)
    o = np.zeros(3)
    lib().orc_rotate(_p(d), ct, phi, _p(o))
    return o


def planck(nu, T):
    return lib().orc_planck(nu, T)


def max_threads():
    return lib().orc_max_threads()
