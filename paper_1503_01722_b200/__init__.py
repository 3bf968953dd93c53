"""Thin Python binding of the C-ABI library `libmc_b200.so` (include/mc.h).

Argument marshalling only: every step of the hot path (source sampling, Woodcock photon transport,
condensed-history electron transport, scoring, batch statistics) runs in the CUDA kernels behind the
C ABI.  There is no CPU path: without the built library the import of any call raises, and without a
CUDA device every compute call returns MC_ERR_CUDA (raised here as McError).

The functions carry the C names (mc_create, mc_build_tables, mc_run, ...).  Output buffers may be
numpy arrays (host) or torch tensors (host or CUDA); PyTorch is used only for device memory and
streams.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmc_b200.so")
_lib = None

MC_OK, MC_ERR_INVALID_ARG, MC_ERR_STATE, MC_ERR_ENERGY_RANGE, MC_ERR_QUEUE_OVERFLOW, MC_ERR_OOM, MC_ERR_CUDA = range(7)
STATUS_NAMES = ["MC_OK", "MC_ERR_INVALID_ARG", "MC_ERR_STATE", "MC_ERR_ENERGY_RANGE", "MC_ERR_QUEUE_OVERFLOW",
                "MC_ERR_OOM", "MC_ERR_CUDA"]
MC_FLAG_NO_HARD_EVENTS, MC_FLAG_NO_MS, MC_FLAG_LOCAL_SECONDARIES = 1, 2, 4
TABLE_IDS = {"mu_tot": 0, "mu_C": 1, "mu_pp": 2, "R": 3, "L": 4, "S_hard": 5, "S_M": 6, "S_max": 7, "K1": 8,
             "mu_maj": 9, "lnA": 10}

# every symbol include/mc.h declares (tests check that the library exports each of them)
SYMBOLS = ["mc_create", "mc_destroy", "mc_build_tables", "mc_export_table", "mc_export_grid", "mc_export_gs_table",
           "mc_set_photon_tables", "mc_run", "mc_run_particles", "mc_run_source", "mc_run_range", "mc_finalize", "mc_edep_buffer",
           "mc_finalize_multi", "mc_finalize_multi_range", "mc_ipc_get_handle", "mc_ipc_open_handle", "mc_ipc_close_handle", "mc_run_atten",
           "mc_edep_total_static", "mc_edep_total_static_max",
           "mc_philox_selftest", "mc_u01_selftest", "mc_bench_red", "mc_bench_issue", "mc_trim", "mc_get_stats", "mc_set_stream", "mc_set_option",
           "mc_last_error", "mc_version"]


class McError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else status}: {msg}")
        self.status = status


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


class _Stats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in (
        "n_histories", "n_electron_steps", "n_photon_flights", "n_fictitious", "n_compton", "n_pair",
        "n_photoelectric", "n_moller", "n_brems", "n_secondary_electrons", "n_secondary_photons",
        "n_dose_atomics", "n_kernel_launches")] + [(n, C.c_double) for n in (
            "e_source_MeV", "e_deposited_MeV", "e_escaped_MeV", "transport_ms", "electron_kernel_ms",
            "photon_kernel_ms")] + [("n_host_syncs", C.c_uint64)]


def lib():
    """The loaded C-ABI library.  Fails loudly if it has not been built (no fallback exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1503_01722_b200.build` "
                              "(this package has no CPU or PyTorch fallback)")
        L = C.CDLL(LIB_PATH)
        vp, u64, i32, u32 = C.c_void_p, C.c_uint64, C.c_int32, C.c_uint32
        L.mc_create.argtypes = [vp, vp, vp, vp, vp, C.POINTER(vp)]
        L.mc_destroy.argtypes = [vp]
        L.mc_destroy.restype = None
        L.mc_build_tables.argtypes = [vp, vp, i32, vp]
        L.mc_export_table.argtypes = [vp, i32, i32, vp]
        L.mc_export_grid.argtypes = [vp, vp]
        L.mc_set_photon_tables.argtypes = [vp, C.c_float, C.c_float, vp, vp, vp, vp]
        L.mc_run.argtypes = [vp, vp, u64, u64, i32, vp, vp]
        L.mc_run_particles.argtypes = [vp, vp, u64, u64, i32, vp, vp]
        L.mc_run_range.argtypes = [vp, vp, u64, u64, u64, u64, i32, vp]
        L.mc_finalize.argtypes = [vp, vp, u64, i32, vp, vp]
        L.mc_edep_buffer.argtypes = [vp, i32, C.POINTER(vp)]
        L.mc_finalize_multi.argtypes = [vp, vp, i32, u64, i32, vp, vp]
        L.mc_finalize_multi_range.argtypes = [vp, vp, i32, u64, i32, C.c_int64, C.c_int64, vp, vp]
        L.mc_ipc_get_handle.argtypes = [vp, vp]
        L.mc_ipc_open_handle.argtypes = [vp, C.POINTER(vp)]
        L.mc_ipc_close_handle.argtypes = [vp]
        L.mc_run_atten.argtypes = [vp, vp, u64, u64, vp, vp]
        L.mc_edep_total_static.argtypes = [vp, u64, vp, vp, vp, i32]
        L.mc_edep_total_static_max.restype = u64
        L.mc_philox_selftest.argtypes = [vp, vp, i32, vp]
        L.mc_bench_red.argtypes = [vp, u32, i32, i32, i32, vp]
        L.mc_bench_issue.argtypes = [vp, i32, vp]
        L.mc_trim.argtypes = [u64]
        L.mc_get_stats.argtypes = [vp, vp]
        L.mc_set_stream.argtypes = [vp, vp]
        L.mc_set_option.argtypes = [vp, C.c_char_p, C.c_int64]
        L.mc_last_error.argtypes = [vp]
        L.mc_last_error.restype = C.c_char_p
        L.mc_version.restype = C.c_char_p
        _lib = L
    return _lib


def _check(ctx, status):
    if status != MC_OK:
        msg = lib().mc_last_error(ctx).decode() if ctx else ""
        raise McError(status, msg)


def _ptr(buf):
    """Raw address of a numpy array or a torch tensor (host or CUDA)."""
    if buf is None:
        return None
    if isinstance(buf, int):
        return buf
    if isinstance(buf, np.ndarray):
        assert buf.flags["C_CONTIGUOUS"]
        return buf.ctypes.data
    assert buf.is_contiguous()
    return buf.data_ptr()


def _beam_struct(beam):
    E = np.ascontiguousarray(beam["E_nodes_MeV"], np.float32)
    p = np.ascontiguousarray(beam["pdf_nodes"], np.float32)
    fp = C.POINTER(C.c_float)
    b = _Beam(int(beam["particle"]), int(beam["shape"]), (C.c_float * 3)(*beam["entry_cm"]),
              (C.c_float * 3)(*beam["axis"]), float(beam["ssd_cm"]), (C.c_float * 2)(*beam["field_cm"]),
              len(E), E.ctypes.data_as(fp), p.ctypes.data_as(fp))
    return b, (E, p)


# ---- the C calls, one Python function each -----------------------------------------------------
def mc_version():
    return lib().mc_version().decode()


def mc_last_error(ctx):
    return lib().mc_last_error(ctx).decode()


def mc_create(material_idx, density_gcc, dims, voxel_cm, origin_cm):
    mat = np.ascontiguousarray(material_idx, np.uint8).reshape(-1)
    rho = np.ascontiguousarray(density_gcc, np.float32).reshape(-1)
    d = np.ascontiguousarray(dims, np.int32)
    assert mat.size == rho.size == int(np.prod(d.astype(np.int64))), "volume size does not match dims"
    h = np.ascontiguousarray(voxel_cm, np.float32)
    o = np.ascontiguousarray(origin_cm, np.float32)
    ctx = C.c_void_p()
    _check(None, lib().mc_create(mat.ctypes.data, rho.ctypes.data, d.ctypes.data, h.ctypes.data, o.ctypes.data,
                                 C.byref(ctx)))
    return ctx


def mc_destroy(ctx):
    lib().mc_destroy(ctx)


def mc_build_tables(ctx, materials, params):
    keep, arr = [], (_Material * len(materials))()
    for i, m in enumerate(materials):
        Z = np.ascontiguousarray(m["Z"], np.int32)
        A = np.ascontiguousarray(m["A"], np.float32)
        w = np.ascontiguousarray(m["w"], np.float32)
        keep += [Z, A, w]
        fp = C.POINTER(C.c_float)
        arr[i] = _Material(len(Z), Z.ctypes.data_as(C.POINTER(C.c_int32)), A.ctypes.data_as(fp),
                           w.ctypes.data_as(fp), m["I_eV"], m["rho_nominal"])
    p = _Params(params["e_cut_MeV"], params["g_cut_MeV"], params["e_max_MeV"], params["n_grid"],
                params["d_maxs_cm"], params["f_maxe"], params["flags"])
    _check(ctx, lib().mc_build_tables(ctx, C.addressof(arr), len(materials), C.addressof(p)))


def mc_export_grid(ctx):
    g = np.zeros(4)
    _check(ctx, lib().mc_export_grid(ctx, g.ctypes.data))
    return {"lnE0": g[0], "dln": g[1], "N": int(g[2]), "k_cut": int(g[3])}


def mc_export_gs_table():
    """The Goudsmit-Saunderson sampling table (R27): (t_nodes[NT], y[NT, NA, NQ] = ln of the quantiles of 1 - cos theta)."""
    dims = (C.c_int32 * 3)()
    _check(None, lib().mc_export_gs_table(dims, None, None))
    t = np.zeros(dims[0], np.float32)
    y = np.zeros((dims[0], dims[1], dims[2]), np.float32)
    _check(None, lib().mc_export_gs_table(dims, t.ctypes.data_as(C.c_void_p), y.ctypes.data_as(C.c_void_p)))
    return t, y


def mc_export_table(ctx, name, material=0):
    N = mc_export_grid(ctx)["N"]
    out = np.zeros(N, np.float32)
    which = TABLE_IDS[name]
    _check(ctx, lib().mc_export_table(ctx, -1 if which == 9 else int(material), which, out.ctypes.data))
    return out


def mc_export_photon_tables(ctx, n_mat):
    """The fp32 photon tables in use, in the dict layout mc_set_photon_tables takes (marshalling only)."""
    g = mc_export_grid(ctx)
    out = {"lnE0": np.float32(g["lnE0"]), "inv_dln": np.float32(1.0 / g["dln"]),
           "mu_maj": mc_export_table(ctx, "mu_maj")}
    for k in ("mu_tot", "mu_C", "mu_pp"):
        out[k] = np.stack([mc_export_table(ctx, k, m) for m in range(n_mat)])
    return out


def mc_set_photon_tables(ctx, tables_f32):
    t = {k: np.ascontiguousarray(tables_f32[k], np.float32) for k in ("mu_maj", "mu_tot", "mu_C", "mu_pp")}
    _check(ctx, lib().mc_set_photon_tables(ctx, C.c_float(tables_f32["lnE0"]), C.c_float(tables_f32["inv_dln"]),
                                           t["mu_maj"].ctypes.data, t["mu_tot"].ctypes.data,
                                           t["mu_C"].ctypes.data, t["mu_pp"].ctypes.data))


def mc_run(ctx, beam, n_histories, seed, n_batches, dose_out, sigma_out):
    b, keep = _beam_struct(beam)
    _check(ctx, lib().mc_run(ctx, C.addressof(b), int(n_histories), int(seed), int(n_batches), _ptr(dose_out),
                             _ptr(sigma_out)))


PARTICLE_DTYPE = np.dtype([("x", "f4"), ("y", "f4"), ("z", "f4"), ("u", "f4"), ("v", "f4"), ("w", "f4"), ("E", "f4"),
                           ("particle", "i4")])  # = mc_particle


def mc_run_particles(ctx, particles, seed, n_batches, dose_out, sigma_out, n=None):
    """particles: numpy structured array of PARTICLE_DTYPE (host) or a CUDA uint8/float tensor holding n such records."""
    if isinstance(particles, np.ndarray):
        particles = np.ascontiguousarray(particles, PARTICLE_DTYPE)
        n = len(particles)
    _check(ctx, lib().mc_run_particles(ctx, _ptr(particles), int(n), int(seed), int(n_batches), _ptr(dose_out),
                                       _ptr(sigma_out)))


SOURCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p)


def mc_run_source(ctx, fn, n, seed, n_batches, dose_out, sigma_out):
    """fn(h_begin, n, out_device_address, cuda_stream) -> 0 on success: writes records h_begin .. h_begin + n - 1 (PARTICLE_DTYPE
    layout) to device memory at out_device_address, with work enqueued on cuda_stream or a blocking copy (marshalling only)."""
    def trampoline(_user, h_begin, cnt, out, stream):
        try:
            return int(fn(int(h_begin), int(cnt), int(out), int(stream or 0)) or 0)
        except Exception:  # noqa: BLE001  (an exception must not cross the C boundary)
            return 1
    cb = SOURCE_FN(trampoline)
    _check(ctx, lib().mc_run_source(ctx, cb, None, C.c_uint64(int(n)), C.c_uint64(int(seed)), int(n_batches), C.c_void_p(_ptr(dose_out)),
                                    C.c_void_p(_ptr(sigma_out))))


def mc_run_range(ctx, beam, n_histories, h_begin, h_end, seed, n_batches, edep_out):
    b, keep = _beam_struct(beam)
    _check(ctx, lib().mc_run_range(ctx, C.addressof(b), int(n_histories), int(h_begin), int(h_end), int(seed),
                                   int(n_batches), _ptr(edep_out)))


def mc_finalize(ctx, edep, n_histories, n_batches, dose_out, sigma_out):
    _check(ctx, lib().mc_finalize(ctx, _ptr(edep), int(n_histories), int(n_batches), _ptr(dose_out), _ptr(sigma_out)))


def mc_edep_buffer(ctx, n_batches):
    """Device address (int) of the context's own [n_batches][nvox] grid buffer."""
    p = C.c_void_p()
    _check(ctx, lib().mc_edep_buffer(ctx, int(n_batches), C.byref(p)))
    return p.value


def mc_finalize_multi(ctx, grids, n_histories, n_batches, dose_out, sigma_out):
    """grids: device addresses (ints) or CUDA tensors, one [n_batches][nvox] grid per rank."""
    addr = [g if isinstance(g, int) else _ptr(g) for g in grids]
    arr = (C.c_void_p * len(addr))(*addr)
    _check(ctx, lib().mc_finalize_multi(ctx, C.addressof(arr), len(addr), int(n_histories), int(n_batches), _ptr(dose_out),
                                        _ptr(sigma_out)))


def mc_finalize_multi_range(ctx, grids, n_histories, n_batches, v_begin, v_end, dose_out, sigma_out):
    """As mc_finalize_multi for voxels [v_begin, v_end): the outputs hold v_end - v_begin floats."""
    addr = [g if isinstance(g, int) else _ptr(g) for g in grids]
    arr = (C.c_void_p * len(addr))(*addr)
    _check(ctx, lib().mc_finalize_multi_range(ctx, C.addressof(arr), len(addr), int(n_histories), int(n_batches), int(v_begin),
                                              int(v_end), _ptr(dose_out), _ptr(sigma_out)))


def mc_ipc_get_handle(dev_ptr):
    h = (C.c_uint8 * 64)()
    _check(None, lib().mc_ipc_get_handle(C.c_void_p(int(dev_ptr)), C.addressof(h)))
    return bytes(h)


def mc_ipc_open_handle(handle):
    h = (C.c_uint8 * 64).from_buffer_copy(handle)
    p = C.c_void_p()
    _check(None, lib().mc_ipc_open_handle(C.addressof(h), C.byref(p)))
    return p.value


def mc_ipc_close_handle(dev_ptr):
    _check(None, lib().mc_ipc_close_handle(C.c_void_p(int(dev_ptr))))


def mc_run_atten(ctx, beam, n, seed, voxel_out, channel_out=None):
    b, keep = _beam_struct(beam)
    _check(ctx, lib().mc_run_atten(ctx, C.addressof(b), int(n), int(seed), _ptr(voxel_out), _ptr(channel_out)))


def mc_edep_total_static_max():
    return int(lib().mc_edep_total_static_max())


def mc_edep_total_static(edep_dev, n, cuda_stream=0, total_out=None):
    """fp64 total of n floats at the device address / CUDA tensor edep_dev, computed without any device allocation
    (include/mc.h).  Returns the total as a float, or writes it to total_out (numpy float64[1] or a CUDA float64 tensor)
    when one is given.  The status message comes back through a caller-owned buffer, as in C."""
    host = np.zeros(1, np.float64)
    msg = C.create_string_buffer(256)
    st = lib().mc_edep_total_static(_ptr(edep_dev), int(n), _ptr(host if total_out is None else total_out),
                                    C.c_void_p(int(cuda_stream)), msg, len(msg))
    if st != MC_OK:
        raise McError(st, msg.value.decode())
    return float(host[0]) if total_out is None else total_out


def mc_philox_selftest(ctr, key):
    ctr = np.ascontiguousarray(ctr, np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, np.uint32).reshape(-1, 2)
    out = np.zeros_like(ctr)
    _check(None, lib().mc_philox_selftest(ctr.ctypes.data, key.ctypes.data, len(ctr), out.ctypes.data))
    return out


def mc_u01_selftest():
    n = C.c_uint64()
    _check(None, lib().mc_u01_selftest(C.byref(n)))
    return int(n.value)


def mc_bench_red(ctx, n_cells, per_thread, mode, blocks):
    ms = C.c_double()
    _check(ctx, lib().mc_bench_red(ctx, int(n_cells), int(per_thread), int(mode), int(blocks), C.addressof(ms)))
    return ms.value


def mc_bench_issue(ctx, iters=4096):
    r = C.c_double()
    _check(ctx, lib().mc_bench_issue(ctx, int(iters), C.addressof(r)))
    return r.value


def mc_trim(keep_bytes=0):
    _check(None, lib().mc_trim(int(keep_bytes)))


def mc_get_stats(ctx):
    s = _Stats()
    _check(ctx, lib().mc_get_stats(ctx, C.addressof(s)))
    return {n: getattr(s, n) for n, _ in _Stats._fields_}


def mc_set_stream(ctx, cuda_stream):
    _check(ctx, lib().mc_set_stream(ctx, C.c_void_p(int(cuda_stream))))


def mc_set_option(ctx, name, value):
    _check(ctx, lib().mc_set_option(ctx, name.encode(), int(value)))


class Engine:
    """Convenience holder of one context: Engine(phantom, materials, params).run(beam, n, seed, B)."""

    def __init__(self, phantom, materials=None, params=None):
        self.nvox = int(np.prod(np.asarray(phantom["dims"], np.int64)))
        self.dims = tuple(int(x) for x in phantom["dims"])
        self.ctx = mc_create(phantom["material"], phantom["density"], phantom["dims"], phantom["voxel_cm"],
                             phantom["origin_cm"])
        if materials is not None:
            mc_build_tables(self.ctx, materials, params)

    def close(self):
        if self.ctx is not None:
            mc_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def run(self, beam, n_histories, seed, n_batches, device_out=False):
        """dose, sigma (MeV/g per history).  device_out=True returns CUDA torch tensors on the current
        torch stream; otherwise host numpy arrays."""
        if device_out:
            import torch
            mc_set_stream(self.ctx, torch.cuda.current_stream().cuda_stream)
            dose = torch.empty(self.nvox, dtype=torch.float32, device="cuda")
            sigma = torch.empty_like(dose)
        else:
            dose, sigma = np.zeros(self.nvox, np.float32), np.zeros(self.nvox, np.float32)
        mc_run(self.ctx, beam, n_histories, seed, n_batches, dose, sigma)
        return dose, sigma

    def stats(self):
        return mc_get_stats(self.ctx)
