"""ctypes harness around the ORACLE (oracle/orc_main.cpp) — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  Nothing under paper_1503_01722_b200/ imports it, and it imports nothing from the CUDA
path (the seeded input generators in paper_1503_01722_b200/workloads.py are handed in by callers).
"""
from __future__ import annotations

import ctypes as C
import multiprocessing as mp
import os

import numpy as np

from . import build as _build

_lib = None

TABLE_IDS = {"mu_tot": 0, "mu_C": 1, "mu_pp": 2, "R": 3, "L": 4, "S_hard": 5, "S_M": 6, "S_max": 7, "K1": 8,
             "mu_maj": 9, "lnA": 10}
STAT_NAMES = ["e_src", "e_dep", "e_esc", "e_cutdep", "n_hist", "n_flight", "n_fict", "n_compton", "n_pair",
              "n_pe", "n_estep", "n_moller", "n_brems", "n_sec_e", "n_sec_g", "path_e", "lim_vox", "lim_maxs",
              "lim_maxe", "lim_range", "lim_event", "max_ledger_rel"]


class _Material(C.Structure):
    _fields_ = [("n_elem", C.c_int32), ("Z", C.POINTER(C.c_int32)), ("A", C.POINTER(C.c_float)),
                ("w", C.POINTER(C.c_float)), ("I_eV", C.c_float), ("rho_nominal", C.c_float)]


class _Params(C.Structure):
    _fields_ = [("e_cut_MeV", C.c_float), ("g_cut_MeV", C.c_float), ("e_max_MeV", C.c_float),
                ("n_grid", C.c_int32), ("d_maxs_cm", C.c_float), ("f_maxe", C.c_float), ("flags", C.c_uint32)]


class _Beam(C.Structure):
    _fields_ = [("particle", C.c_int32), ("shape", C.c_int32), ("entry_cm", C.c_float * 3),
                ("axis", C.c_float * 3), ("ssd_cm", C.c_float), ("field_cm", C.c_float * 2),
                ("n_nodes", C.c_int32), ("E_nodes_MeV", C.POINTER(C.c_float)),
                ("pdf_nodes", C.POINTER(C.c_float))]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_eval.restype = C.c_double
        _lib.orc_eval.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double]
        _lib.orc_lerp.restype = C.c_double
        _lib.orc_lerp.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double]
        _lib.orc_inv_range.restype = C.c_double
        _lib.orc_inv_range.argtypes = [C.c_void_p, C.c_int, C.c_double]
        _lib.orc_material_scalar.restype = C.c_double
        _lib.orc_material_scalar.argtypes = [C.c_void_p, C.c_int, C.c_int]
        _lib.orc_sigma_pp_atom.restype = C.c_double
        _lib.orc_sigma_pp_atom.argtypes = [C.c_int, C.c_double]
        _lib.orc_contract_ln.restype = C.c_float
        _lib.orc_contract_ln.argtypes = [C.c_float]
        _lib.orc_destroy.argtypes = [C.c_void_p]
        _lib.orc_set_flags.argtypes = [C.c_void_p, C.c_uint32]
        _lib.orc_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_double]
        _lib.orc_rotate.argtypes = [C.POINTER(C.c_double), C.c_double, C.c_double, C.POINTER(C.c_double)]
    return _lib


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _beam_struct(beam):
    keep = [np.ascontiguousarray(beam["E_nodes_MeV"], np.float32), np.ascontiguousarray(beam["pdf_nodes"], np.float32)]
    b = _Beam(int(beam["particle"]), int(beam["shape"]), (C.c_float * 3)(*beam["entry_cm"]),
              (C.c_float * 3)(*beam["axis"]), float(beam["ssd_cm"]), (C.c_float * 2)(*beam["field_cm"]),
              len(keep[0]), _fp(keep[0]), _fp(keep[1]))
    return b, keep


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox(c, k, o)
    return [int(x) for x in o]


def contract_ln(x):
    return float(lib().orc_contract_ln(C.c_float(x)))


def sigma_pp_reduced(Z, k):
    """sigma_pair / (alpha r_e^2 Z^2)."""
    return lib().orc_sigma_pp_atom(int(Z), float(k))


class Oracle:
    """One phantom + one set of tables.  Mirrors the C-ABI calls (create / build_tables / run)."""

    def __init__(self, phantom, materials=None, params=None):
        L = lib()
        self._ph = phantom
        self.dims = np.ascontiguousarray(phantom["dims"], np.int32)
        self.nvox = int(np.prod(self.dims))
        self._mat = np.ascontiguousarray(phantom["material"], np.uint8)
        self._rho = np.ascontiguousarray(phantom["density"], np.float32)
        vox = np.ascontiguousarray(phantom["voxel_cm"], np.float32)
        org = np.ascontiguousarray(phantom["origin_cm"], np.float32)
        h = C.c_void_p()
        rc = L.orc_create(self._mat.ctypes.data_as(C.c_void_p), _fp(self._rho),
                          self.dims.ctypes.data_as(C.c_void_p), _fp(vox), _fp(org), C.byref(h))
        if rc:
            raise ValueError(f"orc_create failed ({rc})")
        self._h = h
        self._materials = self._params = None
        if materials is not None:
            self.build_tables(materials, params)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def build_tables(self, materials, params):
        self._materials, self._params = materials, dict(params)
        keep, arr = [], (_Material * len(materials))()
        for i, m in enumerate(materials):
            Z = np.ascontiguousarray(m["Z"], np.int32)
            A = np.ascontiguousarray(m["A"], np.float32)
            w = np.ascontiguousarray(m["w"], np.float32)
            keep += [Z, A, w]
            arr[i] = _Material(len(Z), Z.ctypes.data_as(C.POINTER(C.c_int32)), _fp(A), _fp(w), m["I_eV"],
                               m["rho_nominal"])
        p = _Params(params["e_cut_MeV"], params["g_cut_MeV"], params["e_max_MeV"], params["n_grid"],
                    params["d_maxs_cm"], params["f_maxe"], params["flags"])
        rc = lib().orc_build_tables(self._h, arr, len(materials), C.byref(p))
        if rc:
            raise ValueError(f"orc_build_tables failed ({rc})")

    def set_flags(self, flags):
        self._params["flags"] = int(flags)
        lib().orc_set_flags(self._h, int(flags))

    def set_option(self, name, value):
        """Run-time switches of the readings: hinge_overrun (R8, default 0.25), ms_carry (R8b, default 1)."""
        if lib().orc_set_option(self._h, name.encode(), float(value)):
            raise ValueError(f"orc_set_option({name}, {value}) failed")

    # -- tables / closed forms ---------------------------------------------------------------
    def grid(self):
        o = np.zeros(4)
        lib().orc_grid(self._h, _dp(o))
        return {"lnE0": o[0], "dln": o[1], "N": int(o[2]), "k_cut": int(o[3])}

    def energies(self):
        g = self.grid()
        return np.exp(g["lnE0"] + g["dln"] * np.arange(g["N"]))

    def table(self, name, m=0):
        g = self.grid()
        o = np.zeros(g["N"])
        rc = lib().orc_table(self._h, int(m), TABLE_IDS[name], _dp(o))
        if rc:
            raise ValueError(f"orc_table failed ({rc})")
        return o

    def eval(self, which, E, arg=0.0, m=0):
        ids = {"sigma_kn": 0, "mu_C": 1, "mu_pe": 2, "mu_pp": 3, "L_col": 4, "L_rad": 5, "S_M": 6, "S_br": 7,
               "K1": 8, "delta": 9, "brems_kdsdk": 10, "moller_dsde": 11, "S_el": 12}
        return lib().orc_eval(self._h, int(m), ids[which], float(E), float(arg))

    def lerp(self, name, E, m=0):
        return lib().orc_lerp(self._h, int(m), TABLE_IDS[name], float(E))

    def inv_range(self, Rt, m=0):
        return lib().orc_inv_range(self._h, int(m), float(Rt))

    def material_scalar(self, name, m=0):
        return lib().orc_material_scalar(self._h, int(m), {"ne": 0, "ZA": 1, "Cbr": 2, "Lscr": 3}[name])

    # -- transport ------------------------------------------------------------------------------
    def run_edep(self, beam, n_total, seed, n_batches, h0=0, h1=None, first=False, window=False):
        """Energy deposited per batch grid [B, nvox] (MeV, fp64) for histories [h0, h1) + stats dict.
        first=True also returns (voxel, channel) of each primary photon's first real interaction.
        window=True returns (b_lo, grids[b_lo..b_hi]) — only the batches this history range touches
        (batch of h = floor(h*B/N)); harness-side memory saving, the oracle's arithmetic is unchanged."""
        h1 = n_total if h1 is None else h1
        b, keep = _beam_struct(beam)
        b_lo, b_hi = 0, n_batches - 1
        if window and h1 > h0:
            b_lo, b_hi = (h0 * n_batches) // n_total, ((h1 - 1) * n_batches) // n_total
        edep = np.zeros((b_hi - b_lo + 1, self.nvox))
        st = np.zeros(lib().orc_n_stats())
        fv = np.zeros(h1 - h0, np.int32) if first else None
        fc = np.zeros(h1 - h0, np.int32) if first else None
        # orc_run indexes edep + batch*nvox: hand it the address batch b_lo would have in a full array
        base = C.cast(C.c_void_p(edep.ctypes.data - b_lo * self.nvox * 8), C.POINTER(C.c_double))
        rc = lib().orc_run(self._h, C.byref(b), C.c_uint64(h0), C.c_uint64(h1), C.c_uint64(n_total),
                           C.c_uint64(seed), int(n_batches), base, _dp(st),
                           fv.ctypes.data_as(C.c_void_p) if first else None,
                           fc.ctypes.data_as(C.c_void_p) if first else None)
        if rc:
            raise ValueError(f"orc_run failed ({rc})")
        if window:
            return b_lo, edep, dict(zip(STAT_NAMES, st))
        if first:
            return edep, dict(zip(STAT_NAMES, st)), fv, fc
        return edep, dict(zip(STAT_NAMES, st))

    def run_probe(self, beam, n, seed, h0=0):
        """Per-history probe of the primary electron track (orc_run_probe): dict of arrays + stats."""
        b, keep = _beam_struct(beam)
        npb = lib().orc_n_probe()
        o = np.zeros((n, npb))
        st = np.zeros(lib().orc_n_stats())
        rc = lib().orc_run_probe(self._h, C.byref(b), C.c_uint64(h0), C.c_uint64(h0 + n), C.c_uint64(max(h0 + n, 1)),
                                 C.c_uint64(seed), _dp(o), _dp(st))
        if rc:
            raise ValueError(f"orc_run_probe failed ({rc})")
        out = {"first_hard": o[:, 0].astype(int), "T_first": o[:, 1], "pos": o[:, 2:5], "dir": o[:, 5:8], "path": o[:, 8],
               "steps": o[:, 9], "T_end": o[:, 10], "escaped": o[:, 11].astype(int), "path_first": o[:, 12],
               "fict_before_first": o[:, 13], "q_sampled": o[:, 14], "q_travelled": o[:, 15],
               "annih_sum": o[:, 16:19], "annih_mu": o[:, 19], "brems_cos": o[:, 20], "T_brems": o[:, 21]}
        return out, dict(zip(STAT_NAMES, st))

    def run_particles_edep(self, particles, n_total, seed, n_batches, h0=0, h1=None):
        """Particle-list source: `particles` is a structured array (x, y, z, u, v, w, E float32, particle int32)."""
        h1 = n_total if h1 is None else h1
        pa = np.ascontiguousarray(particles)
        assert pa.dtype.itemsize == 32
        b_lo, b_hi = (h0 * n_batches) // n_total, ((max(h1, h0 + 1) - 1) * n_batches) // n_total
        edep = np.zeros((b_hi - b_lo + 1, self.nvox))
        st = np.zeros(lib().orc_n_stats())
        base = C.cast(C.c_void_p(edep.ctypes.data - b_lo * self.nvox * 8), C.POINTER(C.c_double))
        rc = lib().orc_run_particles(self._h, C.c_void_p(pa.ctypes.data), C.c_uint64(h0), C.c_uint64(h1), C.c_uint64(n_total),
                                     C.c_uint64(seed), int(n_batches), base, _dp(st))
        if rc:
            raise ValueError(f"orc_run_particles failed ({rc})")
        return b_lo, edep, dict(zip(STAT_NAMES, st))

    def run_particles(self, particles, seed, n_batches, workers=1):
        """dose, sigma, stats for a particle list, sharded over `workers` processes by history range."""
        n = len(particles)
        global _FORK_ORC
        edges = np.linspace(0, n, max(1, workers) * 4 + 1).astype(np.int64)
        jobs = [(particles, n, seed, n_batches, int(edges[i]), int(edges[i + 1])) for i in range(len(edges) - 1)
                if edges[i + 1] > edges[i]]
        edep = np.zeros((n_batches, self.nvox))
        stats = []
        if workers <= 1:
            res = [self.run_particles_edep(*j) for j in jobs]
        else:
            _FORK_ORC = self
            try:
                with mp.get_context("fork").Pool(workers) as pool:
                    res = pool.map(_shard_particles, jobs, chunksize=1)
            finally:
                _FORK_ORC = None
        for b_lo, part, st in res:
            edep[b_lo:b_lo + part.shape[0]] += part
            stats.append(st)
        st = {k: (max(r[k] for r in stats) if k == "max_ledger_rel" else sum(r[k] for r in stats)) for k in STAT_NAMES}
        dose, sig = self.finalize(edep, n)
        return dose, sig, st

    def finalize(self, edep, n_total):
        B = edep.shape[0]
        dose, sig = np.zeros(self.nvox), np.zeros(self.nvox)
        lib().orc_finalize(self._h, _dp(np.ascontiguousarray(edep)), C.c_uint64(n_total), int(B), _dp(dose), _dp(sig))
        return dose, sig

    def run(self, beam, n_histories, seed, n_batches, workers=1):
        """dose, sigma (MeV/g per history), stats.  workers>1 shards disjoint history ranges over
        processes (valid because every stream is keyed by the history index)."""
        if workers <= 1:
            edep, st = self.run_edep(beam, n_histories, seed, n_batches)
        else:
            edep, st = _run_sharded(self, beam, n_histories, seed, n_batches, workers)
        dose, sig = self.finalize(edep, n_histories)
        return dose, sig, st

    def run_edep_parallel(self, beam, n_histories, seed, n_batches, workers):
        """run_edep over `workers` processes (disjoint history ranges): edep[B, nvox], stats."""
        if workers <= 1:
            return self.run_edep(beam, n_histories, seed, n_batches)
        return _run_sharded(self, beam, n_histories, seed, n_batches, workers)

    def run_sample(self, beam, n_total, n_sample, seed, n_batches, workers=1):
        """Histories [0, n_sample) of a job of n_total, sharded over `workers` processes: edep[B, nvox],
        stats, wall seconds (the timed CPU baseline of bench.py)."""
        import time
        t0 = time.perf_counter()
        if workers <= 1:
            edep, st = self.run_edep(beam, n_total, seed, n_batches, 0, n_sample)
        else:
            edep, st = _run_sharded(self, beam, n_total, seed, n_batches, workers, h_end=n_sample)
        return edep, st, time.perf_counter() - t0

    def run_atten(self, beam, n, seed, tables_f32):
        """fp32 contract path (R20).  tables_f32: dict(lnE0, inv_dln, mu_maj[N], mu_tot/mu_C/mu_pp[n_mat,N])."""
        b, keep = _beam_struct(beam)
        t = {k: np.ascontiguousarray(tables_f32[k], np.float32) for k in ("mu_maj", "mu_tot", "mu_C", "mu_pp")}
        n_mat, N = t["mu_tot"].shape
        vox = np.zeros(n, np.int32)
        ch = np.zeros(n, np.uint8)
        fl = np.zeros(n, np.uint32)
        rc = lib().orc_run_atten(self._h, C.byref(b), C.c_uint64(n), C.c_uint64(seed), int(N), int(n_mat),
                                 C.c_float(tables_f32["lnE0"]), C.c_float(tables_f32["inv_dln"]),
                                 _fp(t["mu_maj"]), _fp(t["mu_tot"]), _fp(t["mu_C"]), _fp(t["mu_pp"]),
                                 vox.ctypes.data_as(C.c_void_p), ch.ctypes.data_as(C.c_void_p),
                                 fl.ctypes.data_as(C.c_void_p))
        if rc:
            raise ValueError(f"orc_run_atten failed ({rc})")
        return vox, ch, fl

    def photon_tables_f32(self):
        """The oracle's own photon tables rounded to fp32, in the layout run_atten takes."""
        g = self.grid()
        nm = len(self._materials)
        out = {"lnE0": np.float32(g["lnE0"]), "inv_dln": np.float32(1.0 / g["dln"]),
               "mu_maj": self.table("mu_maj").astype(np.float32)}
        for k in ("mu_tot", "mu_C", "mu_pp"):
            out[k] = np.stack([self.table(k, m) for m in range(nm)]).astype(np.float32)
        return out

    def sample_source(self, beam, n, seed):
        b, keep = _beam_struct(beam)
        o = np.zeros((n, 7))
        lib().orc_sample_source(self._h, C.byref(b), C.c_uint64(n), C.c_uint64(seed), _dp(o))
        return o

    def sample_brems(self, T0, n, seed, m=0):
        o = np.zeros(n)
        lib().orc_sample_brems(self._h, int(m), C.c_double(T0), C.c_uint64(n), C.c_uint64(seed), _dp(o))
        return o


def sample_kn(E, n, seed=1):
    o = np.zeros((n, 4))
    lib().orc_sample_kn(C.c_double(E), C.c_uint64(n), C.c_uint64(seed), _dp(o))
    return o


def sample_moller(T0, e_cut, n, seed=1):
    o = np.zeros((n, 3))
    lib().orc_sample_moller(C.c_double(T0), C.c_double(e_cut), C.c_uint64(n), C.c_uint64(seed), _dp(o))
    return o


def sample_iso(n, seed=1):
    o = np.zeros((n, 3))
    lib().orc_sample_iso(C.c_uint64(n), C.c_uint64(seed), _dp(o))
    return o


def rotate(d, mu, phi):
    """The transport code's direction rotation (R25): d rotated by polar cosine mu and azimuth phi."""
    di = (C.c_double * 3)(*[float(x) for x in d])
    o = (C.c_double * 3)()
    lib().orc_rotate(di, float(mu), float(phi), o)
    return np.array(o[:])


# -- Goudsmit-Saunderson multiple scattering (orc_gs.h; R27) -----------------------------------------
def gs_dims():
    o = (C.c_int * 3)()
    lib().orc_gs_dims(o)
    return tuple(o)


def gs_nodes():
    nt, na, nq = gs_dims()
    t, A, r = np.zeros(nt), np.zeros(na), np.zeros(nq)
    lib().orc_gs_nodes(_dp(t), _dp(A), _dp(r))
    return t, A, r


def gs_table():
    """ln of the quantiles of 1 - cos(theta): [NT, NA, NQ]."""
    nt, na, nq = gs_dims()
    o = np.zeros((nt, na, nq))
    lib().orc_gs_table(_dp(o))
    return o


def gs_moments(A, lmax):
    o = np.zeros(lmax + 1)
    lib().orc_gs_moments(C.c_double(A), int(lmax), _dp(o))
    return o


def gs_G1(A):
    lib().orc_gs_G1.restype = C.c_double
    return lib().orc_gs_G1(C.c_double(A))


def gs_cdf(lam, A, x):
    x = np.ascontiguousarray(x, np.float64)
    o = np.zeros(len(x))
    lib().orc_gs_cdf(C.c_double(lam), C.c_double(A), _dp(x), int(len(x)), _dp(o))
    return o


def gs_sample(t, A, n, seed=1):
    """n samples of cos(theta) from the table sampler transport uses."""
    o = np.zeros(n)
    lib().orc_gs_sample(C.c_double(t), C.c_double(A), C.c_uint64(n), C.c_uint64(seed), _dp(o))
    return o


def sample_ms(a, n, seed=1):
    o = np.zeros(n)
    lib().orc_sample_ms(C.c_double(a), C.c_uint64(n), C.c_uint64(seed), _dp(o))
    return o


# -- sharding over host cores -------------------------------------------------------------------
_FORK_ORC = None  # the parent's Oracle, inherited by forked workers (tables are built once, not per chunk)


def _shard_particles(args):
    return _FORK_ORC.run_particles_edep(*args)


def _shard(args):
    beam, n_total, seed, B, h0, h1 = args
    return _FORK_ORC.run_edep(beam, n_total, seed, B, h0, h1, window=True)


def _run_sharded(orc, beam, n_total, seed, B, workers, h_end=None):
    # many small contiguous chunks so that every worker ends at about the same time; a chunk returns
    # only the batch grids its history range touches
    global _FORK_ORC
    n_chunks = workers * 8
    edges = np.linspace(0, n_total if h_end is None else h_end, n_chunks + 1).astype(np.int64)
    jobs = [(beam, n_total, seed, B, int(edges[i]), int(edges[i + 1])) for i in range(n_chunks)
            if edges[i + 1] > edges[i]]
    _FORK_ORC = orc
    edep = np.zeros((B, orc.nvox))
    stats = []
    try:
        with mp.get_context("fork").Pool(workers) as pool:
            for b_lo, part, st in pool.imap_unordered(_shard, jobs, chunksize=1):
                edep[b_lo:b_lo + part.shape[0]] += part
                stats.append(st)
    finally:
        _FORK_ORC = None
    st = {k: (max(r[k] for r in stats) if k == "max_ledger_rel" else sum(r[k] for r in stats)) for k in STAT_NAMES}
    return edep, st


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1
