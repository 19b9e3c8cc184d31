"""Thin ctypes binding of the C-ABI CUDA library (include/pyjac_b200.h).

Argument marshalling only: every step of the evaluation runs in the library's sm_100a kernels.
PyTorch is used for device memory and streams.  There is no CPU fallback: a missing library or a
failing CUDA call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .mechanism import Mechanism

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpyjac_b200.so")
TOOLS_LIB_PATH = os.path.join(_HERE, "libpyjac_b200_tools.so")     # include/pyjac_b200_tools.h: bench / test helpers

PYJAC_OK, PYJAC_EINVAL, PYJAC_ENOMEM, PYJAC_ECUDA, PYJAC_ELIMIT, PYJAC_ESCRATCH = 0, -1, -2, -3, -4, -5

_pd = C.POINTER(C.c_double)
_pi = C.POINTER(C.c_int32)


class MechDesc(C.Structure):
    """struct pyjac_mech_desc"""
    _fields_ = [("n_species", C.c_int32), ("n_reactions", C.c_int32),
                ("mol_wt", _pd), ("nasa_lo", _pd), ("nasa_hi", _pd), ("t_mid", _pd),
                ("reac_ptr", _pi), ("reac_spec", _pi), ("reac_nu", _pi),
                ("prod_ptr", _pi), ("prod_spec", _pi), ("prod_nu", _pi),
                ("rxn_type", _pi), ("rev_type", _pi),
                ("arr_hi", _pd), ("arr_lo", _pd), ("arr_rev", _pd),
                ("falloff_form", _pi), ("falloff_par", _pd), ("tb_species", _pi),
                ("eff_ptr", _pi), ("eff_spec", _pi), ("eff_val", _pd),
                ("plog_ptr", _pi), ("plog_p", _pd), ("plog_arr", _pd),
                ("cheb_ptr", _pi), ("cheb_nT", _pi), ("cheb_nP", _pi),
                ("cheb_lim", _pd), ("cheb_eta", _pd)]


class LaunchShape(C.Structure):
    """struct pyjac_launch_shape (0 = let the library choose)"""
    _fields_ = [("states_per_cta", C.c_int32), ("threads", C.c_int32), ("ctas_per_sm", C.c_int32),
                ("list_cap", C.c_int32), ("cell_cap", C.c_int32), ("rows_per_lane", C.c_int32),
                ("p1_states", C.c_int32), ("stage_tables", C.c_int32), ("layout", C.c_int32)]


EXPORTS = ("pyjac_mech_create", "pyjac_mech_create_shaped", "pyjac_mech_create_error", "pyjac_mech_destroy", "pyjac_mech_trim",
           "pyjac_mech_sizes",
           "pyjac_eval_rates", "pyjac_eval_dydt", "pyjac_eval_jacobian", "pyjac_eval_jacobian_host",
           "pyjac_eval_dydt_host", "pyjac_eval_jvp", "pyjac_eval_jacobian_fd", "pyjac_fd_workspace_doubles",
           "pyjac_eval_jacobian_fd_static", "pyjac_fd_static_max_states", "pyjac_kernel_launches",
           "pyjac_jacobian_launch_config", "pyjac_strerror")
TOOLS_EXPORTS = ("pyjac_tools_pack_stats", "pyjac_tools_peak_store_stream", "pyjac_tools_peak_tile_store",
                 "pyjac_tools_peak_dfma", "pyjac_tools_gather_probe")

_lib = None
_tools = None


def load_library(path: str | None = None):
    """Loads libpyjac_b200.so (built in-tree by `python -m paper_1605_03262_b200.build`)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise RuntimeError("%s is missing: run `python -m paper_1605_03262_b200.build` "
                           "(there is no CPU fallback)" % p)
    lib = C.CDLL(p)
    vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int32
    lib.pyjac_mech_create.argtypes = [C.POINTER(MechDesc), C.c_int, C.POINTER(vp)]
    lib.pyjac_mech_create_shaped.argtypes = [C.POINTER(MechDesc), C.c_int, C.POINTER(LaunchShape), C.POINTER(vp)]
    lib.pyjac_mech_destroy.argtypes = [vp]
    lib.pyjac_mech_trim.argtypes = [vp]
    lib.pyjac_mech_sizes.argtypes = [vp, C.POINTER(i32), C.POINTER(i32)]
    lib.pyjac_eval_rates.argtypes = [vp, i64, vp, vp, vp, i64, vp, vp, vp, vp, vp]
    lib.pyjac_eval_dydt.argtypes = [vp, i64, vp, vp, vp, i64, vp, vp]
    lib.pyjac_eval_jacobian.argtypes = [vp, i64, vp, vp, vp, i64, vp, vp]
    lib.pyjac_eval_jacobian_host.argtypes = [vp, i64, vp, vp, vp, i64, vp, i64]
    lib.pyjac_eval_dydt_host.argtypes = [vp, i64, vp, vp, vp, i64, vp, i64]
    lib.pyjac_eval_jvp.argtypes = [vp, i64, vp, vp, vp, i64, vp, i64, vp, vp]
    lib.pyjac_eval_jacobian_fd.argtypes = [vp, i64, vp, vp, vp, i64, C.c_double, C.c_double, vp, vp, i64, vp]
    lib.pyjac_fd_workspace_doubles.argtypes = [vp, i64]
    lib.pyjac_fd_workspace_doubles.restype = i64
    lib.pyjac_eval_jacobian_fd_static.argtypes = [vp, i64, vp, vp, vp, i64, C.c_double, C.c_double, vp, vp]
    lib.pyjac_fd_static_max_states.argtypes = [vp]
    lib.pyjac_fd_static_max_states.restype = i64
    lib.pyjac_kernel_launches.argtypes = []
    lib.pyjac_kernel_launches.restype = i64
    lib.pyjac_jacobian_launch_config.argtypes = [vp, i64] + [C.POINTER(i32)] * 5
    lib.pyjac_strerror.argtypes = [C.c_int]
    lib.pyjac_strerror.restype = C.c_char_p
    lib.pyjac_mech_create_error.argtypes = []
    lib.pyjac_mech_create_error.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("pyjac_kernel_launches", "pyjac_strerror", "pyjac_mech_create_error", "pyjac_fd_workspace_doubles",
                        "pyjac_fd_static_max_states"):
            getattr(lib, name).restype = C.c_int
    if path is None:
        _lib = lib
    return lib


def load_tools(path: str | None = None):
    """Loads libpyjac_b200_tools.so (table statistics, machine-peak probes; not the product)."""
    global _tools
    if _tools is not None and path is None:
        return _tools
    p = path or TOOLS_LIB_PATH
    if not os.path.exists(p):
        raise RuntimeError("%s is missing: run `python -m paper_1605_03262_b200.build`" % p)
    lib = C.CDLL(p)
    vp, i64 = C.c_void_p, C.c_int64
    lib.pyjac_tools_pack_stats.argtypes = [C.POINTER(MechDesc), C.POINTER(LaunchShape), C.POINTER(i64)]
    lib.pyjac_tools_peak_store_stream.argtypes = [vp, i64, vp]
    lib.pyjac_tools_peak_dfma.argtypes = [vp, i64, C.POINTER(i64), vp]
    lib.pyjac_tools_peak_tile_store.argtypes = [vp, i64, C.c_int32, C.c_int32, C.c_int32, vp]
    lib.pyjac_tools_gather_probe.argtypes = [C.POINTER(MechDesc), C.c_int32, C.c_int32, C.c_int32, C.c_int32, i64, vp,
                                             _pd, C.POINTER(i64), C.c_int32, C.POINTER(C.c_float), C.POINTER(C.c_float), vp]
    for name in TOOLS_EXPORTS:
        getattr(lib, name).restype = C.c_int
    if path is None:
        _tools = lib
    return lib


class PyJacError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        lib = load_library()
        msg = lib.pyjac_strerror(code).decode()
        if what.startswith("pyjac_mech_create"):
            why = lib.pyjac_mech_create_error().decode()
            msg = msg + (": " + why if why else "")
        super().__init__("%s failed: %s (%d)" % (what, msg, code))


def _check(code, what):
    if code != PYJAC_OK:
        raise PyJacError(code, what)


def mech_desc(mech: Mechanism):
    """(MechDesc, keepalive) for a `Mechanism` (host arrays, C layout)."""
    m = mech.normalized()
    d = MechDesc()
    d.n_species, d.n_reactions = m.n_species, m.n_reactions
    keep = []
    for dst, src in (("mol_wt", "mol_wt"), ("nasa_lo", "nasa_lo"), ("nasa_hi", "nasa_hi"),
                     ("t_mid", "t_mid"), ("arr_hi", "arr_hi"), ("arr_lo", "arr_lo"),
                     ("arr_rev", "arr_rev"), ("falloff_par", "falloff_par"), ("eff_val", "eff_val"),
                     ("plog_p", "plog_p"), ("plog_arr", "plog_arr"), ("cheb_lim", "cheb_lim"),
                     ("cheb_eta", "cheb_eta")):
        a = np.ascontiguousarray(getattr(m, src), dtype=np.float64)
        keep.append(a)
        setattr(d, dst, a.ctypes.data_as(_pd))
    for name in ("reac_ptr", "reac_spec", "reac_nu", "prod_ptr", "prod_spec", "prod_nu", "rxn_type",
                 "rev_type", "falloff_form", "tb_species", "eff_ptr", "eff_spec", "plog_ptr",
                 "cheb_ptr", "cheb_nT", "cheb_nP"):
        a = np.ascontiguousarray(getattr(m, name), dtype=np.int32)
        keep.append(a)
        setattr(d, name, a.ctypes.data_as(_pi))
    return d, keep


def launch_shape(shape):
    """None, a LaunchShape or a dict with the fields of `pyjac_launch_shape` -> LaunchShape or None."""
    if shape is None or isinstance(shape, LaunchShape):
        return shape
    unknown = set(shape) - {f[0] for f in LaunchShape._fields_}
    if unknown:
        raise ValueError("unknown launch-shape fields: %s" % sorted(unknown))
    return LaunchShape(**{k: int(v) for k, v in shape.items()})


PACK_STAT_NAMES = ("e_elements", "cell_entries", "b_steps", "a_steps", "cells", "chunks",
                   "smem_bytes_per_cta", "reaction_groups", "states_per_cta", "threads", "reserved10",
                   "ctas_per_sm_target", "heavy_cells", "heavy_pieces", "a_table_bytes", "b_table_bytes",
                   "a_steps_sum3", "a_steps_sum1", "a_steps_prod", "a_steps_all3", "a_conflict_wf", "b_conflict_wf",
                   "layout_excess_before", "layout_excess_after")


def pack_stats(mech: Mechanism, shape=None) -> dict:
    """Host-only (tools library): sizes of the evaluation tables `pyjac_mech_create_shaped` would build."""
    lib = load_tools()
    d, keep = mech_desc(mech)
    out = (C.c_int64 * len(PACK_STAT_NAMES))()
    sh = launch_shape(shape)
    _check(lib.pyjac_tools_pack_stats(C.byref(d), C.byref(sh) if sh is not None else None, out), "pyjac_tools_pack_stats")
    return dict(zip(PACK_STAT_NAMES, [int(v) for v in out]))


def peak_store_stream(buf, stream_ptr):
    """Enqueues one write-only pass over the CUDA float64 tensor `buf` (pyjac_tools_peak_store_stream)."""
    _check(load_tools().pyjac_tools_peak_store_stream(buf.data_ptr(), int(buf.numel()), stream_ptr),
           "pyjac_tools_peak_store_stream")


def peak_tile_store(buf, n_tiles, tile_doubles, mode, ctas_per_sm, stream_ptr):
    """Enqueues the tile-store probe on the CUDA float64 tensor `buf` (pyjac_tools_peak_tile_store): mode 0 one bulk
    copy per tile, mode 1 shared-memory read-back and streaming stores."""
    if buf.numel() < int(n_tiles) * int(tile_doubles):
        raise ValueError("buf is too small for n_tiles tiles")
    _check(load_tools().pyjac_tools_peak_tile_store(buf.data_ptr(), int(n_tiles), int(tile_doubles), int(mode),
                                                    int(ctas_per_sm), stream_ptr), "pyjac_tools_peak_tile_store")


def gather_probe(mech: Mechanism, out, n_states, S, threads, ctas_per_sm, n_buf, reps, stream_ptr) -> dict:
    """Runs the gather probe of the tools library (pyjac_tools_gather_probe: unpadded, length-balanced gathers into a
    per-state shared-memory tile + one bulk copy per state; timing prototype on the mechanism's real cell lists) and
    returns its timings, table statistics and the expected tile."""
    d, keep = mech_desc(mech)
    ld = mech.n_species + 1
    if out.numel() < int(n_states) * ld * ld:
        raise ValueError("out is too small")
    expected = np.empty(ld * ld)
    stats = (C.c_int64 * 8)()
    best, mean = C.c_float(), C.c_float()
    _check(load_tools().pyjac_tools_gather_probe(C.byref(d), int(S), int(threads), int(ctas_per_sm), int(n_buf), int(n_states),
                                                 out.data_ptr(), expected.ctypes.data_as(_pd), stats, int(reps),
                                                 C.byref(best), C.byref(mean), stream_ptr), "pyjac_tools_gather_probe")
    names = ("entries", "entries_padded", "chunks", "e_elements", "smem_bytes", "nonempty_cells", "cells", "grid")
    return dict(ms_best=best.value, ms_mean=mean.value, expected=expected, **dict(zip(names, [int(v) for v in stats])))


def peak_dfma(out, iters, stream_ptr):
    """Enqueues the fp64 FMA probe (pyjac_tools_peak_dfma); returns the flops it executes."""
    n = C.c_int64()
    _check(load_tools().pyjac_tools_peak_dfma(out.data_ptr(), int(iters), C.byref(n), stream_ptr), "pyjac_tools_peak_dfma")
    return 2 * 8 * int(iters) * n.value


class PyJac:
    """A kinetic model resident on one CUDA device (wraps `pyjac_mech*`)."""

    def __init__(self, mech: Mechanism, device: int = 0, shape=None):
        self.lib = load_library()
        d, keep = mech_desc(mech)
        h = C.c_void_p()
        sh = launch_shape(shape)
        if sh is None:
            _check(self.lib.pyjac_mech_create(C.byref(d), int(device), C.byref(h)), "pyjac_mech_create")
        else:
            _check(self.lib.pyjac_mech_create_shaped(C.byref(d), int(device), C.byref(sh), C.byref(h)),
                   "pyjac_mech_create_shaped")
        self._h = h
        self.device = int(device)
        ns, nr = C.c_int32(), C.c_int32()
        _check(self.lib.pyjac_mech_sizes(h, C.byref(ns), C.byref(nr)), "pyjac_mech_sizes")
        self.ns, self.nr = ns.value, nr.value

    def close(self):
        if getattr(self, "_h", None):
            self.lib.pyjac_mech_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- helpers
    def _dev_inputs(self, T, P, Y):
        import torch
        for t in (T, P, Y):
            if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64):
                raise TypeError("T, P, Y must be float64 CUDA tensors")
        if Y.dim() != 2 or Y.stride(1) != 1 or not T.is_contiguous() or not P.is_contiguous():
            raise ValueError("Y must be [n][>=Nsp] with unit inner stride; T, P contiguous")
        if any(t.device.index != self.device for t in (T, P, Y)):
            raise ValueError("T, P, Y must live on the handle's device (cuda:%d)" % self.device)
        n = T.numel()
        if P.numel() != n or Y.shape[0] != n or Y.shape[1] < self.ns:
            raise ValueError("inconsistent state arrays")
        import torch
        if torch.cuda.current_device() != self.device:
            raise ValueError("the current CUDA device (whose stream the call is enqueued on) is not cuda:%d" % self.device)
        ldy = Y.stride(0) if n > 1 else max(Y.shape[1], self.ns)
        return n, ldy

    @staticmethod
    def _stream():
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)

    def _dev_out(self, out, n, per_state, like):
        """A caller's output tensor is written in place: it must be a contiguous float64 CUDA tensor on the
        handle's device with at least n * per_state elements (nothing is ever copied or converted)."""
        import torch
        if out is None:
            return torch.empty((n, per_state), dtype=torch.float64, device=like.device)
        if not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.is_contiguous()
                and out.device.index == self.device and out.numel() >= n * per_state):
            raise ValueError("out must be a contiguous float64 CUDA tensor on cuda:%d with at least %d elements"
                             % (self.device, n * per_state))
        return out

    # ---- device-pointer calls (enqueue on torch's current stream)
    def eval_rates(self, T, P, Y, want=("rf", "rr", "cmod", "wdot"), out=None):
        """dict of float64 CUDA tensors rf, rr, cmod [n][Nreac], wdot [n][Nsp] (pyjac_eval_rates).  `out`: a dict of
        caller-owned tensors to write in place (its keys are the outputs wanted; nothing is allocated then)."""
        import torch
        n, ldy = self._dev_inputs(T, P, Y)
        if out is not None:
            if set(out) - {"rf", "rr", "cmod", "wdot"}:
                raise ValueError("unknown rate outputs: %s" % sorted(set(out) - {"rf", "rr", "cmod", "wdot"}))
            out = {k: self._dev_out(v, n, self.ns if k == "wdot" else self.nr, T) for k, v in out.items()}
        else:
            out = {}
            for name in ("rf", "rr", "cmod", "wdot"):
                if name in want:
                    out[name] = torch.empty((n, self.ns if name == "wdot" else self.nr),
                                            dtype=torch.float64, device=T.device)
        ptr = lambda k: C.c_void_p(out[k].data_ptr()) if k in out else None
        _check(self.lib.pyjac_eval_rates(self._h, n, T.data_ptr(), P.data_ptr(), Y.data_ptr(), ldy,
                                         ptr("rf"), ptr("rr"), ptr("cmod"), ptr("wdot"),
                                         self._stream()), "pyjac_eval_rates")
        return out

    def eval_dydt(self, T, P, Y, out=None):
        """[n][Nsp+1] source term (pyjac_eval_dydt)."""
        import torch
        n, ldy = self._dev_inputs(T, P, Y)
        out = self._dev_out(out, n, self.ns + 1, T)
        _check(self.lib.pyjac_eval_dydt(self._h, n, T.data_ptr(), P.data_ptr(), Y.data_ptr(), ldy,
                                        out.data_ptr(), self._stream()), "pyjac_eval_dydt")
        return out

    def eval_jacobian(self, T, P, Y, out=None):
        """[n][(Nsp+1)^2] column-major Jacobians (pyjac_eval_jacobian)."""
        import torch
        n, ldy = self._dev_inputs(T, P, Y)
        ld = self.ns + 1
        out = self._dev_out(out, n, ld * ld, T)
        _check(self.lib.pyjac_eval_jacobian(self._h, n, T.data_ptr(), P.data_ptr(), Y.data_ptr(), ldy,
                                            out.data_ptr(), self._stream()), "pyjac_eval_jacobian")
        return out

    def eval_jvp(self, T, P, Y, v, out=None):
        """[n][Nsp+1] Jacobian-vector products J v, one vector v[n][>= Nsp+1] per state (pyjac_eval_jvp): the
        matrix is never formed."""
        import torch
        n, ldy = self._dev_inputs(T, P, Y)
        ld = self.ns + 1
        if (not isinstance(v, torch.Tensor) or not v.is_cuda or v.dtype != torch.float64 or v.dim() != 2
                or v.shape[0] != n or v.shape[1] < ld or v.stride(1) != 1 or v.device != T.device):
            raise ValueError("v must be a float64 CUDA tensor [n][>= Nsp+1] with unit inner stride on the inputs' device")
        out = self._dev_out(out, n, ld, T)
        ldv = v.stride(0) if n > 1 else max(v.shape[1], ld)
        _check(self.lib.pyjac_eval_jvp(self._h, n, T.data_ptr(), P.data_ptr(), Y.data_ptr(), ldy, v.data_ptr(),
                                       int(ldv), out.data_ptr(), self._stream()), "pyjac_eval_jvp")
        return out

    def fd_workspace_doubles(self, chunk_states: int) -> int:
        return int(self.lib.pyjac_fd_workspace_doubles(self._h, int(chunk_states)))

    def eval_jacobian_fd(self, T, P, Y, out=None, rtol: float = 1e-8, atol: float = 1e-15, work=None,
                         chunk_states: int = 4096):
        """First-order forward-difference Jacobians from the source term (pyjac_eval_jacobian_fd), same layout
        as eval_jacobian.  `work`: a float64 CUDA tensor of scratch (default: one for `chunk_states` states)."""
        import torch
        n, ldy = self._dev_inputs(T, P, Y)
        ld = self.ns + 1
        out = self._dev_out(out, n, ld * ld, T)
        if work is None:
            work = torch.empty(self.fd_workspace_doubles(max(1, min(int(chunk_states), n))), dtype=torch.float64,
                               device=T.device)
        if not work.is_cuda or work.dtype != torch.float64 or not work.is_contiguous() or work.device != T.device:
            raise ValueError("work must be a contiguous float64 CUDA tensor on the inputs' device")
        _check(self.lib.pyjac_eval_jacobian_fd(self._h, n, T.data_ptr(), P.data_ptr(), Y.data_ptr(), ldy,
                                               float(rtol), float(atol), out.data_ptr(), work.data_ptr(),
                                               int(work.numel()), self._stream()), "pyjac_eval_jacobian_fd")
        return out

    def fd_static_max_states(self) -> int:
        """Largest batch eval_jacobian_fd_static takes for this mechanism (pyjac_fd_static_max_states)."""
        return int(self.lib.pyjac_fd_static_max_states(self._h))

    def eval_jacobian_fd_static(self, T, P, Y, out, rtol: float = 1e-8, atol: float = 1e-15):
        """eval_jacobian_fd for callers that cannot allocate device memory (pyjac_eval_jacobian_fd_static): an
        application whose own arena already owns the whole GPU, or a callback in a time-step loop that must not
        trigger cudaMalloc's device-wide synchronisation.  The scratch is a 32 MiB array built into the library, so
        `out` is required (nothing is allocated here either) and at most fd_static_max_states() states go in one
        call; more raises PyJacError with code PYJAC_ESCRATCH.  One array per GPU is shared by all calls: keep calls
        ordered on one stream.  The first call on a device does a one-time address lookup on the host."""
        n, ldy = self._dev_inputs(T, P, Y)
        ld = self.ns + 1
        if out is None:
            raise ValueError("eval_jacobian_fd_static allocates nothing: pass `out`")
        out = self._dev_out(out, n, ld * ld, T)
        _check(self.lib.pyjac_eval_jacobian_fd_static(self._h, n, T.data_ptr(), P.data_ptr(), Y.data_ptr(), ldy,
                                                      float(rtol), float(atol), out.data_ptr(), self._stream()),
               "pyjac_eval_jacobian_fd_static")
        return out

    # ---- host-pointer calls (copies inside; synchronous)
    @staticmethod
    def _host_in(a):
        """Host input: a CPU float64 torch tensor or anything numpy can view as C-contiguous float64 (inputs
        may be converted; the converted copy is kept alive for the call)."""
        import torch
        if isinstance(a, torch.Tensor):
            if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous():
                raise ValueError("host inputs must be contiguous float64 CPU tensors")
            return a.data_ptr(), a
        a = np.ascontiguousarray(a, dtype=np.float64)
        return a.ctypes.data, a

    @staticmethod
    def _host_out(a, n_elements):
        """Host output, written in place: never copied or converted, so it must already be C-contiguous float64
        with room for the result."""
        import torch
        if isinstance(a, torch.Tensor):
            if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or a.numel() < n_elements:
                raise ValueError("out must be a contiguous float64 CPU tensor with at least %d elements" % n_elements)
            return a.data_ptr()
        if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
                and a.flags["WRITEABLE"] and a.size >= n_elements):
            raise ValueError("out must be a writeable C-contiguous float64 numpy array with at least %d elements"
                             % n_elements)
        return a.ctypes.data

    def _host_call(self, fn, what, T, P, Y, out, per_state, chunk_states):
        (pT, kT), (pP, kP), (pY, kY) = map(self._host_in, (T, P, Y))
        n = int(kT.shape[0])
        if kY.ndim != 2 or int(kY.shape[0]) != n or int(kP.shape[0]) != n or int(kY.shape[1]) < self.ns:
            raise ValueError("inconsistent state arrays")
        pO = self._host_out(out, n * per_state)
        _check(fn(self._h, n, pT, pP, pY, int(kY.shape[1]), pO, int(chunk_states)), what)
        return out

    def eval_jacobian_host(self, T, P, Y, out, chunk_states: int = 0):
        """Host buffers in, host buffer out (numpy arrays or CPU torch tensors, pinned or not)."""
        ld = self.ns + 1
        return self._host_call(self.lib.pyjac_eval_jacobian_host, "pyjac_eval_jacobian_host", T, P, Y, out, ld * ld,
                               chunk_states)

    def eval_dydt_host(self, T, P, Y, out, chunk_states: int = 0):
        return self._host_call(self.lib.pyjac_eval_dydt_host, "pyjac_eval_dydt_host", T, P, Y, out, self.ns + 1,
                               chunk_states)

    def trim(self):
        """Frees the device staging buffers the *_host calls keep with the handle (pyjac_mech_trim)."""
        _check(self.lib.pyjac_mech_trim(self._h), "pyjac_mech_trim")

    def launch_config(self, n: int):
        v = [C.c_int32() for _ in range(5)]
        _check(self.lib.pyjac_jacobian_launch_config(self._h, int(n), *[C.byref(x) for x in v]),
               "pyjac_jacobian_launch_config")
        return dict(threads=v[0].value, smem_bytes=v[1].value, ctas_per_sm=v[2].value, grid=v[3].value,
                    states_per_cta=v[4].value)

    def kernel_launches(self) -> int:
        return int(self.lib.pyjac_kernel_launches())
