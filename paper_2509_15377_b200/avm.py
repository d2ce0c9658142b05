"""Thin ctypes binding of libavm (include/avm.h): argument marshalling only — every step of the path runs in
the CUDA kernels of csrc/.  Function names follow the C ABI without the `avm_` prefix (avm.run <-> avm_run).

PyTorch is used for device memory (torch.empty(..., device="cuda")), the stream handle and nothing else.
There is no CPU fallback: importing this module without a built libavm.so raises ImportError.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.environ.get("AVM_LIBRARY") or os.path.join(_HERE, "libavm.so")    # AVM_LIBRARY: the -DAVM_DEBUG build (build.SO_DEBUG)
if not os.path.exists(_SO):
    raise ImportError(f"{_SO} is missing: build it with `python -m paper_2509_15377_b200.build` "
                      "(nvcc, sm_100a).  There is no CPU fallback.")
_lib = C.CDLL(_SO)

OK, ERR_INVALID_ARG, ERR_CAPACITY, ERR_CUDA, ERR_STATE = 0, -1, -2, -3, -4
RUN_PRIMARIES_ON_DEVICE, RUN_SHAPE_WIDE, RUN_SHAPE_LATENCY, RUN_BANDED = 1, 4, 8, 16
MAX_LEVELS, MAX_SLABS = 64, 8
RUN_STATIC_MAX_CAPACITY = 65536     # AVM_RUN_STATIC_MAX_CAPACITY: largest `capacity` run_static accepts
EXPORTS = ["avm_last_error", "avm_ctx_create", "avm_ctx_destroy", "avm_ctx_sm_count", "avm_gas_bytes",
           "avm_gas_create", "avm_gas_destroy", "avm_gas_nu_hat", "avm_gas_bands", "avm_field_create", "avm_field_destroy", "avm_tetmesh_bytes",
           "avm_field_eval", "avm_run_workspace_bytes", "avm_run", "avm_run_static", "avm_run_static_bytes", "avm_run_stats", "avm_run_transport_ms", "avm_fetch", "avm_ion_drift", "avm_step_batch", "avm_step_batch_form",
           "avm_philox_batch", "avm_fp64_probe", "avm_gather_probe", "avm_smem_probe"]


class AvmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"avm error {code}: {msg}")
        self.code = code


class _GasDesc(C.Structure):
    _fields_ = [("n_bins", C.c_int32), ("e_max_eV", C.c_double), ("n_levels", C.c_int32),
                ("cum_rate", C.c_void_p), ("level_type", C.c_void_p), ("level_loss_eV", C.c_void_p),
                ("level_recoil", C.c_void_p), ("level_ob_w_eV", C.c_void_p), ("nu_hat", C.c_double),
                ("scat_xi", C.c_void_p), ("level_penning_prob", C.c_void_p), ("level_penning_eV", C.c_void_p),
                ("kT_eV", C.c_double)]


class _Slab(C.Structure):
    _fields_ = [("z_lo", C.c_double), ("z_hi", C.c_double), ("kind", C.c_int32), ("E", C.c_double * 3),
                ("nodes_dev", C.c_void_p), ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("origin", C.c_double * 3), ("spacing", C.c_double * 3), ("bc_x", C.c_int32), ("bc_y", C.c_int32),
                ("period_x", C.c_double), ("period_y", C.c_double), ("nodes_f64_dev", C.c_void_p),
                ("n_mesh_nodes", C.c_int64), ("n_tets", C.c_int64), ("node_xyz", C.c_void_p), ("node_V", C.c_void_p),
                ("tet_nodes", C.c_void_p), ("tet_gas", C.c_void_p), ("mesh_dev", C.c_void_p), ("mesh_dev_bytes", C.c_size_t)]


class _FieldDesc(C.Structure):
    _fields_ = [("slabs", C.POINTER(_Slab)), ("n_slabs", C.c_int32), ("B", C.c_double * 3),
                ("xy_lo", C.c_double * 2), ("xy_hi", C.c_double * 2)]


class _Signal(C.Structure):
    _fields_ = [("weighting", C.c_void_p), ("t0", C.c_double), ("dt_bin", C.c_double), ("n_bins", C.c_int32),
                ("signal_dev", C.c_void_p)]


class _IonOpts(C.Structure):
    _fields_ = [("mobility_pos", C.c_double), ("mobility_neg", C.c_double), ("step_cm", C.c_double), ("t_max", C.c_double),
                ("max_steps", C.c_int32)]


class _RunOpts(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("t_max", C.c_double), ("flags", C.c_uint32),
                ("max_iters_per_launch", C.c_uint32), ("id_offset", C.c_uint64), ("max_ctas", C.c_int32),
                ("signal", C.POINTER(_Signal))]


class _Outputs(C.Structure):
    _fields_ = [("capacity", C.c_int64), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("id", C.c_void_p), ("avalanche", C.c_void_p), ("status", C.c_void_p), ("n_steps", C.c_void_p),
                ("birth", C.c_void_p), ("end", C.c_void_p), ("per_avalanche", C.c_void_p),
                ("tallies_u64", C.c_void_p), ("tallies_f64", C.c_void_p)]


_lib.avm_last_error.restype = C.c_char_p
_lib.avm_gas_bytes.restype = C.c_size_t
_lib.avm_tetmesh_bytes.restype = C.c_size_t
_lib.avm_tetmesh_bytes.argtypes = [C.c_void_p]
_lib.avm_run_workspace_bytes.restype = C.c_size_t
_lib.avm_run_workspace_bytes.argtypes = [C.c_void_p, C.c_int64]
_lib.avm_gas_nu_hat.restype = C.c_double
_lib.avm_gas_nu_hat.argtypes = [C.c_void_p]
for _n in ("avm_ctx_create", "avm_ctx_destroy", "avm_ctx_sm_count", "avm_gas_create", "avm_gas_destroy", "avm_gas_bands",
           "avm_field_create", "avm_field_destroy", "avm_field_eval", "avm_run", "avm_run_stats", "avm_fetch", "avm_ion_drift",
           "avm_step_batch", "avm_step_batch_form", "avm_philox_batch", "avm_fp64_probe", "avm_run_transport_ms",
           "avm_gather_probe", "avm_smem_probe"):
    getattr(_lib, _n).restype = C.c_int32
_lib.avm_run_transport_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
_lib.avm_ctx_create.argtypes = [C.c_int32, C.c_void_p, C.POINTER(C.c_void_p)]
_lib.avm_ctx_destroy.argtypes = [C.c_void_p]
_lib.avm_ctx_sm_count.argtypes = [C.c_void_p]
_lib.avm_gas_create.argtypes = [C.c_void_p, C.POINTER(_GasDesc), C.c_void_p, C.c_size_t, C.POINTER(C.c_void_p)]
_lib.avm_gas_destroy.argtypes = [C.c_void_p]
_lib.avm_gas_bands.argtypes = [C.c_void_p] + [C.c_void_p] * 4
_lib.avm_field_create.argtypes = [C.c_void_p, C.POINTER(_FieldDesc), C.POINTER(C.c_void_p)]
_lib.avm_field_destroy.argtypes = [C.c_void_p]
_lib.avm_field_eval.argtypes = [C.c_void_p, C.c_void_p, C.c_int64] + [C.c_void_p] * 4
_lib.avm_run.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(_RunOpts),
                         C.POINTER(_Outputs), C.POINTER(C.c_int64)]
_lib.avm_run_static.restype = C.c_int32
_lib.avm_run_static.argtypes = list(_lib.avm_run.argtypes)
_lib.avm_run_static_bytes.restype = C.c_size_t
_lib.avm_run_static_bytes.argtypes = []
_lib.avm_ion_drift.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_Signal), C.POINTER(_IonOpts), C.POINTER(_Outputs), C.c_int64, C.c_int64,
                               C.c_void_p, C.c_void_p, C.c_void_p]
_lib.avm_run_stats.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
_lib.avm_fetch.argtypes = [C.c_void_p, C.POINTER(_Outputs), C.c_int64, C.c_int64, C.c_int32, C.POINTER(_Outputs)]
_lib.avm_step_batch.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64, C.c_double, C.c_int64] + [C.c_void_p] * 9
_lib.avm_step_batch_form.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64, C.c_double, C.c_int32, C.c_int32, C.c_int64] + [C.c_void_p] * 9 + [C.c_uint32]
_lib.avm_philox_batch.argtypes = [C.c_void_p, C.c_uint64, C.c_int64] + [C.c_void_p] * 5
_lib.avm_gather_probe.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_int32, C.c_int32, C.c_int64, C.c_void_p, C.POINTER(C.c_float)]
_lib.avm_smem_probe.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int64, C.c_void_p, C.POINTER(C.c_float)]
_lib.avm_fp64_probe.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_void_p, C.POINTER(C.c_float)]


def last_error() -> str:
    return _lib.avm_last_error().decode()


def _check(rc, allow=()):
    if rc != OK and rc not in allow:
        raise AvmError(rc, last_error())
    return rc


def _hp(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _dev(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


class Context:
    """avm_ctx: a device ordinal and the CUDA stream all work is enqueued on."""

    def __init__(self, device: int = 0, stream: Optional[torch.cuda.Stream] = None):
        if not torch.cuda.is_available():
            raise AvmError(ERR_CUDA, "no CUDA device visible; libavm has no CPU fallback")
        self.device = torch.device("cuda", device)
        self.stream = stream
        handle = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream(self.device).cuda_stream)
        self._h = C.c_void_p()
        _check(_lib.avm_ctx_create(device, handle, C.byref(self._h)))

    @property
    def sm_count(self) -> int:
        return int(_lib.avm_ctx_sm_count(self._h))

    def empty(self, shape, dtype):
        return torch.empty(shape, dtype=dtype, device=self.device)

    def close(self):
        if self._h:
            _lib.avm_ctx_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def ctx_create(device: int = 0, stream=None) -> Context:
    return Context(device, stream)


class Gas:
    """avm_gas: rate tables resident on the device (buffer owned here, borrowed by the library)."""

    def __init__(self, ctx: Context, table):
        self.ctx = ctx
        cum = np.ascontiguousarray(table.cum_rate, dtype=np.float64)
        ty = np.ascontiguousarray(table.level_type, dtype=np.uint8)
        lo = np.ascontiguousarray(table.level_loss, dtype=np.float64)
        rc = np.ascontiguousarray(table.level_recoil, dtype=np.float64)
        w = np.ascontiguousarray(table.level_ob_w, dtype=np.float64)
        self.n_levels = int(cum.shape[1])
        self.n_bins = int(cum.shape[0])
        opt = [None if getattr(table, k, None) is None else np.ascontiguousarray(getattr(table, k), dtype=np.float64)
               for k in ("scat_xi", "level_penning_prob", "level_penning_eV")]              # NEXT-3 extensions (optional)
        d = _GasDesc(self.n_bins, float(table.e_max), self.n_levels, _hp(cum).value, _hp(ty).value, _hp(lo).value,
                     _hp(rc).value, _hp(w).value, float(table.nu_hat), *[None if a is None else _hp(a).value for a in opt],
                     float(getattr(table, "kT_eV", 0.0)))
        nbytes = int(_lib.avm_gas_bytes(C.byref(d)))
        if nbytes == 0:
            raise AvmError(ERR_INVALID_ARG, "gas: invalid description")
        self.buf = ctx.empty(nbytes, torch.uint8)
        self._h = C.c_void_p()
        _check(_lib.avm_gas_create(ctx._h, C.byref(d), _dev(self.buf), nbytes, C.byref(self._h)))
        self.nbytes = nbytes

    @property
    def nu_hat(self) -> float:
        return float(_lib.avm_gas_nu_hat(self._h))

    def bands(self):
        """avm_gas_bands: (a2 [J], nu [K, J+1], dtmax [K, J+1], shift) — the table of banded null-collision rates."""
        shp = np.zeros(3, dtype=np.int32)
        _check(_lib.avm_gas_bands(self._h, _hp(shp), None, None, None))
        K, J, shift = (int(v) for v in shp)
        a2 = np.zeros(J); nu = np.zeros((K, J + 1)); dt = np.zeros((K, J + 1))
        _check(_lib.avm_gas_bands(self._h, _hp(shp), _hp(a2), _hp(nu), _hp(dt)))
        return a2, nu, dt, shift

    def __del__(self):
        try:
            if self._h:
                _lib.avm_gas_destroy(self._h)
        except Exception:
            pass


def gas_create(ctx, table) -> Gas:
    return Gas(ctx, table)


class Field:
    """avm_field: slab descriptors; grid nodes are uploaded once into torch device tensors kept alive here
    (the one-off field-map transfer the paper excludes from its timings)."""

    def __init__(self, ctx: Context, desc, widen: bool = True):
        """widen: also give the library an fp64 scratch copy of every grid map (avm_slab.nodes_f64_dev): twice the
        bytes, no float-to-double conversions in the lookup; results are identical."""
        self.ctx = ctx
        n = len(desc.slabs)
        arr = (_Slab * max(n, 1))()
        self.nodes = []
        self.wide = []
        self.map_bytes = 0
        for i, s in enumerate(desc.slabs):
            a = arr[i]
            a.z_lo, a.z_hi, a.kind = s.z_lo, s.z_hi, s.kind
            a.E[:] = s.E
            if s.nodes is not None:
                if isinstance(s.nodes, torch.Tensor):
                    t = s.nodes.to(device=ctx.device, dtype=torch.float32).contiguous()
                else:
                    t = torch.from_numpy(np.ascontiguousarray(s.nodes, dtype=np.float32)).to(ctx.device)
                self.nodes.append(t)
                self.map_bytes += t.numel() * 4
                a.nodes_dev = t.data_ptr()
                a.nz, a.ny, a.nx = t.shape[:3]
                if widen:
                    wd = torch.empty(t.numel(), dtype=torch.float64, device=ctx.device)
                    self.wide.append(wd)
                    a.nodes_f64_dev = wd.data_ptr()
            a.origin[:] = s.origin
            a.spacing[:] = s.spacing
            a.bc_x, a.bc_y, a.period_x, a.period_y = s.bc_x, s.bc_y, s.period_x, s.period_y
            m = getattr(s, "mesh", None)
            if m is not None:                   # kind 2: host arrays in, device buffer sized by the library (NEXT-2)
                host = [np.ascontiguousarray(m.node_xyz, dtype=np.float64), np.ascontiguousarray(m.node_V, dtype=np.float64),
                        np.ascontiguousarray(m.tet_nodes, dtype=np.int32), np.ascontiguousarray(m.tet_gas, dtype=np.uint8)]
                self.nodes.append(host)
                a.n_mesh_nodes, a.n_tets = host[0].shape[0], host[2].shape[0]
                a.node_xyz, a.node_V, a.tet_nodes, a.tet_gas = (_hp(x).value for x in host)
                nbytes = int(_lib.avm_tetmesh_bytes(C.byref(a)))
                if nbytes == 0:
                    raise AvmError(ERR_INVALID_ARG, "field: invalid mesh: " + last_error())
                buf = ctx.empty(nbytes, torch.uint8)
                self.wide.append(buf)
                self.map_bytes += nbytes
                a.mesh_dev, a.mesh_dev_bytes = buf.data_ptr(), nbytes
        d = _FieldDesc(arr, n, (C.c_double * 3)(*desc.B), (C.c_double * 2)(*desc.xy_lo), (C.c_double * 2)(*desc.xy_hi))
        self._h = C.c_void_p()
        _check(_lib.avm_field_create(ctx._h, C.byref(d), C.byref(self._h)))

    def __del__(self):
        try:
            if self._h:
                _lib.avm_field_destroy(self._h)
        except Exception:
            pass


def field_create(ctx, desc, widen: bool = True) -> Field:
    return Field(ctx, desc, widen)


def field_eval(ctx: Context, field: Field, r):
    """r: [3, n] (numpy or cuda tensor) -> E [3, n], mask [n], slab [n] as numpy."""
    rt = torch.as_tensor(np.ascontiguousarray(r, dtype=np.float64)).to(ctx.device) if not isinstance(r, torch.Tensor) else r.contiguous()
    n = rt.shape[1]
    E = ctx.empty((3, n), torch.float64); m = ctx.empty(n, torch.float64); sl = ctx.empty(n, torch.int32)
    _check(_lib.avm_field_eval(ctx._h, field._h, n, _dev(rt), _dev(E), _dev(m), _dev(sl)))
    return E.cpu().numpy(), m.cpu().numpy(), sl.cpu().numpy()


@dataclass
class StepResult:
    state: np.ndarray
    event: np.ndarray
    status: np.ndarray
    bin: np.ndarray
    child: np.ndarray
    child_id: np.ndarray


def step_batch(ctx: Context, gas: Gas, field: Field, seed, state, ids, n_idx, t_max=float("inf")) -> StepResult:
    st = torch.from_numpy(np.ascontiguousarray(state, dtype=np.float64)).to(ctx.device)
    n = st.shape[1]
    idt = torch.from_numpy(np.ascontiguousarray(ids, dtype=np.uint64).view(np.int64)).to(ctx.device)
    nt = torch.from_numpy(np.ascontiguousarray(n_idx, dtype=np.uint32).view(np.int32)).to(ctx.device)
    out = ctx.empty((8, n), torch.float64); ev = ctx.empty(n, torch.int32); stt = ctx.empty(n, torch.int32)
    bn = ctx.empty(n, torch.int32); ch = ctx.empty((8, n), torch.float64); cid = ctx.empty(n, torch.int64)
    _check(_lib.avm_step_batch(ctx._h, gas._h, field._h, int(seed), float(t_max), n, _dev(st), _dev(idt), _dev(nt),
                               _dev(out), _dev(ev), _dev(stt), _dev(bn), _dev(ch), _dev(cid)))
    return StepResult(out.cpu().numpy(), ev.cpu().numpy(), stt.cpu().numpy(), bn.cpu().numpy(), ch.cpu().numpy(),
                      cid.cpu().numpy().view(np.uint64))


def step_form_lanes(k: int) -> int:
    """Steps per time-parallel batch when a warp holds k electrons: 32 / 2^ceil(log2 k)."""
    return 32 >> max(int(k) - 1, 0).bit_length()


def step_batch_form(ctx: Context, gas: Gas, field: Field, seed, state, ids, n_idx, form: int, k: int = 1,
                    t_max=float("inf"), flags: int = 0) -> StepResult:
    """avm_step_batch_form.  Forms 0 / 1: as step_batch.  Forms 2 / 3: arrays get a trailing axis of gl =
    step_form_lanes(k) steps per electron ([8, n, gl], [n, gl]); steps the batch did not reach have event == -3."""
    st = torch.from_numpy(np.ascontiguousarray(state, dtype=np.float64)).to(ctx.device)
    n = st.shape[1]
    gl = step_form_lanes(k) if form >= 2 else 1
    m = n * gl
    idt = torch.from_numpy(np.ascontiguousarray(ids, dtype=np.uint64).view(np.int64)).to(ctx.device)
    nt = torch.from_numpy(np.ascontiguousarray(n_idx, dtype=np.uint32).view(np.int32)).to(ctx.device)
    out = torch.zeros((8, m), dtype=torch.float64, device=ctx.device)
    ev = torch.full((m,), -3, dtype=torch.int32, device=ctx.device)
    stt = torch.zeros(m, dtype=torch.int32, device=ctx.device)
    bn = torch.full((m,), -1, dtype=torch.int32, device=ctx.device)
    ch = torch.zeros((8, m), dtype=torch.float64, device=ctx.device)
    cid = torch.zeros(m, dtype=torch.int64, device=ctx.device)
    _check(_lib.avm_step_batch_form(ctx._h, gas._h, field._h, int(seed), float(t_max), int(form), int(k), n, _dev(st),
                                    _dev(idt), _dev(nt), _dev(out), _dev(ev), _dev(stt), _dev(bn), _dev(ch), _dev(cid),
                                    int(flags)))
    r = StepResult(out.cpu().numpy(), ev.cpu().numpy(), stt.cpu().numpy(), bn.cpu().numpy(), ch.cpu().numpy(),
                   cid.cpu().numpy().view(np.uint64))
    if form >= 2:
        r = StepResult(r.state.reshape(8, n, gl), r.event.reshape(n, gl), r.status.reshape(n, gl), r.bin.reshape(n, gl),
                       r.child.reshape(8, n, gl), r.child_id.reshape(n, gl))
    return r


def philox_batch(ctx: Context, seed, ids, n_idx, block):
    idt = torch.from_numpy(np.ascontiguousarray(ids, dtype=np.uint64).view(np.int64)).to(ctx.device)
    n = idt.shape[0]
    nt = torch.from_numpy(np.ascontiguousarray(n_idx, dtype=np.uint32).view(np.int32)).to(ctx.device)
    bt = torch.from_numpy(np.ascontiguousarray(block, dtype=np.uint32).view(np.int32)).to(ctx.device)
    w = ctx.empty((n, 4), torch.int32); u = ctx.empty((n, 2), torch.float64)
    _check(_lib.avm_philox_batch(ctx._h, int(seed), n, _dev(idt), _dev(nt), _dev(bt), _dev(w), _dev(u)))
    return w.cpu().numpy().view(np.uint32), u.cpu().numpy()


def fp64_probe(ctx: Context, n_blocks=None, n_threads=256, iters=1 << 16) -> dict:
    """Measured FP64 FMA issue rate of the device (thread-instructions per second)."""
    nb = n_blocks or ctx.sm_count * 8
    sink = ctx.empty(nb * n_threads, torch.float64)
    ms = C.c_float(0)
    _check(_lib.avm_fp64_probe(ctx._h, nb, n_threads, iters, _dev(sink), C.byref(ms)))
    n_fma = float(nb) * n_threads * iters * 8
    return {"ms": ms.value, "dfma_per_s": n_fma / (ms.value * 1e-3), "threads": nb * n_threads}


def gather_probe(ctx: Context, working_set_bytes: int, iters: int = 2048, blocks_per_sm: int = 8, n_threads: int = 256) -> dict:
    """Measured random 32-byte-sector gather bandwidth over a working set of the given size (L2-resident or HBM)."""
    buf = torch.zeros(int(working_set_bytes) // 8, dtype=torch.int64, device=ctx.device)
    nb = ctx.sm_count * blocks_per_sm
    sink = ctx.empty(nb * n_threads, torch.int64)
    ms = C.c_float(0)
    _check(_lib.avm_gather_probe(ctx._h, _dev(buf), buf.numel() * 8, nb, n_threads, iters, _dev(sink), C.byref(ms)))
    moved = float(nb) * n_threads * iters * 32
    return {"ms": ms.value, "GBps": moved / (ms.value * 1e-3) / 1e9, "sectors_per_s": moved / 32 / (ms.value * 1e-3),
            "working_set_bytes": int(buf.numel() * 8)}


def smem_probe(ctx: Context, table_bytes: int = 160000, iters: int = 1 << 14, n_threads: int = 512) -> dict:
    """Measured shared-memory random 8-byte loads per second, one CTA per SM."""
    nb = ctx.sm_count
    sink = ctx.empty(nb * n_threads, torch.int64)
    ms = C.c_float(0)
    _check(_lib.avm_smem_probe(ctx._h, int(table_bytes), nb, n_threads, iters, _dev(sink), C.byref(ms)))
    return {"ms": ms.value, "loads_per_s": float(nb) * n_threads * iters / (ms.value * 1e-3)}


class RunBuffers:
    """Caller-side device buffers of avm_outputs for a given capacity (allocated once, reused by runs)."""

    def __init__(self, ctx: Context, capacity: int, n_primaries: int, n_levels: int):
        self.ctx, self.capacity, self.n_primaries, self.n_levels = ctx, int(capacity), int(n_primaries), int(n_levels)
        cap = self.capacity
        self.ws_bytes = int(_lib.avm_run_workspace_bytes(ctx._h, cap))
        self.workspace = ctx.empty(self.ws_bytes, torch.uint8)
        self.id = ctx.empty(cap, torch.int64)
        self.avalanche = ctx.empty(cap, torch.int32)
        self.status = ctx.empty(cap, torch.int32)
        self.n_steps = ctx.empty(cap, torch.int32)
        self.birth = ctx.empty((5, cap), torch.float64)
        self.end = ctx.empty((8, cap), torch.float64)
        self.per_avalanche = ctx.empty((max(self.n_primaries, 1), 3), torch.int64)
        self.tallies_u64 = ctx.empty(n_levels + 5, torch.int64)
        self.tallies_f64 = ctx.empty(5, torch.float64)

    def c_struct(self) -> _Outputs:
        return _Outputs(self.capacity, _dev(self.workspace), self.ws_bytes, _dev(self.id), _dev(self.avalanche),
                        _dev(self.status), _dev(self.n_steps), _dev(self.birth), _dev(self.end),
                        _dev(self.per_avalanche), _dev(self.tallies_u64), _dev(self.tallies_f64))


class HostBuffers:
    """Host mirror of RunBuffers for avm_fetch (pinned when possible)."""

    def __init__(self, capacity: int, n_primaries: int, n_levels: int, pinned: bool = True):
        self.capacity, self.n_primaries, self.n_levels = int(capacity), int(n_primaries), int(n_levels)
        cap = self.capacity

        def mk(shape, dtype):
            return torch.empty(shape, dtype=dtype, pin_memory=pinned)
        self.id = mk(cap, torch.int64); self.avalanche = mk(cap, torch.int32); self.status = mk(cap, torch.int32)
        self.n_steps = mk(cap, torch.int32); self.birth = mk((5, cap), torch.float64); self.end = mk((8, cap), torch.float64)
        self.per_avalanche = mk((max(self.n_primaries, 1), 3), torch.int64)
        self.tallies_u64 = mk(n_levels + 5, torch.int64); self.tallies_f64 = mk(5, torch.float64)

    def c_struct(self) -> _Outputs:
        p = lambda t: C.c_void_p(t.data_ptr())
        return _Outputs(self.capacity, None, 0, p(self.id), p(self.avalanche), p(self.status), p(self.n_steps),
                        p(self.birth), p(self.end), p(self.per_avalanche), p(self.tallies_u64), p(self.tallies_f64))


@dataclass
class RunResult:
    n: int
    id: np.ndarray
    avalanche: np.ndarray
    status: np.ndarray
    n_steps: np.ndarray
    birth: np.ndarray           # [5, n]
    end: np.ndarray             # [8, n]
    per_avalanche: np.ndarray   # [Np, 3]
    tallies_u64: np.ndarray     # [L+5]: per level, null, real, overflow, steps, Penning transfers
    tallies_f64: np.ndarray     # [5]
    rc: int = 0

    def sorted_by_id(self):
        o = np.argsort(self.id, kind="stable")
        return RunResult(self.n, self.id[o], self.avalanche[o], self.status[o], self.n_steps[o], self.birth[:, o],
                         self.end[:, o], self.per_avalanche, self.tallies_u64, self.tallies_f64, self.rc)


def _signal_struct(signal):
    """signal = (weighting Field, t0, dt_bin, float64 CUDA tensor [n_bins]) -> avm_signal (or None)."""
    if signal is None:
        return None
    wf, t0, dt_bin, arr = signal
    assert arr.is_cuda and arr.dtype == torch.float64 and arr.is_contiguous()
    return _Signal(wf._h, float(t0), float(dt_bin), int(arr.numel()), arr.data_ptr())


def run(ctx: Context, gas: Gas, field: Field, primaries, bufs: RunBuffers, seed=0, t_max=float("inf"), flags=0,
        max_iters_per_launch=0, id_offset=0, max_ctas=0, allow_overflow=False, signal=None) -> tuple:
    """avm_run.  primaries: numpy/CPU tensor [Np, 8] (H2D inside the call) or a CUDA tensor (flag set here).
    signal: None or (weighting Field, t0, dt_bin, float64 CUDA tensor [n_bins], added to) — the induced signal (NEXT-4).
    Returns (rc, n_endpoints); outputs stay in `bufs` on the device."""
    if isinstance(primaries, torch.Tensor) and primaries.is_cuda:
        p = primaries.contiguous()
        assert p.dtype == torch.float64
        flags |= RUN_PRIMARIES_ON_DEVICE
        ptr, np_ = C.c_void_p(p.data_ptr()), p.shape[0]
    elif isinstance(primaries, torch.Tensor):
        p = primaries.contiguous()
        assert p.dtype == torch.float64
        ptr, np_ = C.c_void_p(p.data_ptr()), p.shape[0]
    else:
        p = np.ascontiguousarray(primaries, dtype=np.float64)
        ptr, np_ = _hp(p), p.shape[0]
    sg = _signal_struct(signal)
    opts = _RunOpts(int(seed), float(t_max), int(flags), int(max_iters_per_launch), int(id_offset), int(max_ctas),
                    C.pointer(sg) if sg is not None else None)
    o = bufs.c_struct()
    n_out = C.c_int64(0)
    rc = _lib.avm_run(ctx._h, gas._h, field._h, ptr, np_, C.byref(opts), C.byref(o), C.byref(n_out))
    _check(rc, allow=(ERR_CAPACITY,) if allow_overflow else ())
    return rc, int(n_out.value)


def run_static_bytes() -> int:
    """avm_run_static_bytes: size of the scratch block built into libavm.so (held by every GPU that loads it)."""
    return int(_lib.avm_run_static_bytes())


def run_static(ctx: Context, gas: Gas, field: Field, primaries, bufs: RunBuffers, seed=0, t_max=float("inf"), flags=0,
               max_iters_per_launch=0, id_offset=0, max_ctas=0, allow_overflow=False, signal=None) -> tuple:
    """avm_run_static: the same run as `run`, for callers that cannot allocate device memory for a workspace (a plug-in
    whose host framework owns the allocator, a service with a memory pool frozen at start-up).  The transport kernel's
    scratch lives in a fixed block inside the library instead, so `bufs.workspace` is not passed at all (NULL / 0 go
    down); inputs and outputs are still the caller's tensors.  Limit: bufs.capacity <= RUN_STATIC_MAX_CAPACITY (65536
    electrons), beyond it the call raises AvmError (INVALID_ARG) and nothing runs.  One block per GPU, shared by every
    call: calls from several host threads to one GPU must be serialised by the caller.  The first call on a device looks
    the block's address up; make it outside any stream capture.  Returns (rc, n_endpoints) like `run`."""
    if isinstance(primaries, torch.Tensor) and primaries.is_cuda:
        p = primaries.contiguous()
        assert p.dtype == torch.float64
        flags |= RUN_PRIMARIES_ON_DEVICE
        ptr, np_ = C.c_void_p(p.data_ptr()), p.shape[0]
    elif isinstance(primaries, torch.Tensor):
        p = primaries.contiguous()
        assert p.dtype == torch.float64
        ptr, np_ = C.c_void_p(p.data_ptr()), p.shape[0]
    else:
        p = np.ascontiguousarray(primaries, dtype=np.float64)
        ptr, np_ = _hp(p), p.shape[0]
    sg = _signal_struct(signal)
    opts = _RunOpts(int(seed), float(t_max), int(flags), int(max_iters_per_launch), int(id_offset), int(max_ctas),
                    C.pointer(sg) if sg is not None else None)
    o = bufs.c_struct()
    o.workspace, o.workspace_bytes = None, 0          # ignored by the entry point; passed as NULL to show it
    n_out = C.c_int64(0)
    rc = _lib.avm_run_static(ctx._h, gas._h, field._h, ptr, np_, C.byref(opts), C.byref(o), C.byref(n_out))
    _check(rc, allow=(ERR_CAPACITY,) if allow_overflow else ())
    return rc, int(n_out.value)


def run_stats(ctx: Context) -> tuple:
    a, b = C.c_int64(0), C.c_int64(0)
    _check(_lib.avm_run_stats(ctx._h, C.byref(a), C.byref(b)))
    return int(a.value), int(b.value)


def run_transport_ms(ctx: Context) -> float:
    ms = C.c_float(0)
    _check(_lib.avm_run_transport_ms(ctx._h, C.byref(ms)))
    return float(ms.value)


def fetch(ctx: Context, bufs: RunBuffers, n: int, host: Optional[HostBuffers] = None) -> RunResult:
    """avm_fetch: device -> host copy of the first n endpoints and the tallies.  With caller-provided `host` buffers the
    result holds VIEWS into them (valid until they are reused: no second copy on the host); without, views into buffers
    of its own."""
    host = host or HostBuffers(max(n, 1), bufs.n_primaries, bufs.n_levels, pinned=False)
    d, h = bufs.c_struct(), host.c_struct()
    _check(_lib.avm_fetch(ctx._h, C.byref(d), n, bufs.n_primaries, bufs.n_levels, C.byref(h)))
    u64 = lambda t: t.numpy().view(np.uint64)      # numpy views keep their torch storage alive
    return RunResult(n, u64(host.id)[:n], host.avalanche.numpy().view(np.uint32)[:n], host.status.numpy()[:n],
                     host.n_steps.numpy().view(np.uint32)[:n], host.birth.numpy()[:, :n], host.end.numpy()[:, :n],
                     u64(host.per_avalanche)[:bufs.n_primaries], u64(host.tallies_u64), host.tallies_f64.numpy())


@dataclass
class IonResult:
    end: np.ndarray        # [4, 2n]: x, y, z, t; entry s = positive ion born with electron s, n + s = negative ion of electron s
    status: np.ndarray     # [2n]; -1 = no such ion
    n_steps: np.ndarray


def ion_drift(ctx: Context, field: Field, bufs: RunBuffers, n: int, mobility_pos, mobility_neg, step_cm, t_max=float("inf"),
              max_steps=1 << 20, signal=None) -> IonResult:
    """avm_ion_drift on the outputs of a finished run (still on the device in `bufs`)."""
    ie = ctx.empty((4, 2 * max(n, 1)), torch.float64); ist = ctx.empty(2 * max(n, 1), torch.int32); ins = ctx.empty(2 * max(n, 1), torch.int32)
    sg = _signal_struct(signal)
    io = _IonOpts(float(mobility_pos), float(mobility_neg), float(step_cm), float(t_max), int(max_steps))
    o = bufs.c_struct()
    _check(_lib.avm_ion_drift(ctx._h, field._h, C.byref(sg) if sg is not None else None, C.byref(io), C.byref(o), int(n),
                              int(bufs.n_primaries), _dev(ie), _dev(ist), _dev(ins)))
    torch.cuda.synchronize(ctx.device)
    return IonResult(ie.cpu().numpy()[:, :2 * n], ist.cpu().numpy()[:2 * n], ins.cpu().numpy().view(np.uint32)[:2 * n])


def simulate(ctx: Context, gas: Gas, field: Field, primaries, seed=0, t_max=float("inf"), capacity=None, **kw) -> RunResult:
    """Convenience for tests: allocate buffers, avm_run with host primaries, avm_fetch."""
    prim = np.ascontiguousarray(primaries, dtype=np.float64)
    cap = int(capacity if capacity is not None else max(4 * prim.shape[0], 1 << 16))
    bufs = RunBuffers(ctx, cap, prim.shape[0], gas.n_levels)
    rc, n = run(ctx, gas, field, prim, bufs, seed=seed, t_max=t_max, **kw)
    res = fetch(ctx, bufs, n)
    res.rc = rc
    return res
