"""ctypes binding of the ORACLE (oracle/avmo.cpp).  TEST INFRASTRUCTURE: imported only by tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs — never by the product package.

`build()` compiles oracle/libavmo.so with g++ -O2 -ffp-contract=off (building the checker is not using it).
Inputs are the plain-data descriptions of paper_2509_15377_b200.gen (GasTable, FieldDesc) and numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO_SAN = os.path.join(_HERE, "libavmo_san.so")        # build(sanitize=True): the same source under ASan + UBSan
# AVMO_SANITIZED=1 makes this process load the sanitizer build (the process must then run with libasan preloaded:
# tests/test_oracle_sanitizers.py does that in a subprocess)
_SANITIZED = os.environ.get("AVMO_SANITIZED") == "1"
_SO = _SO_SAN if _SANITIZED else os.path.join(_HERE, "libavmo.so")
_lib = None


def build(force: bool = False, sanitize: bool = _SANITIZED) -> str:
    """sanitize: -fsanitize=address,undefined (the oracle under ASan / UBSan), every report fatal."""
    src = os.path.join(_HERE, "avmo.cpp")
    hdr = os.path.join(_HERE, "avmo.h")
    so = _SO_SAN if sanitize else os.path.join(_HERE, "libavmo.so")
    if not force and os.path.exists(so) and os.path.getmtime(so) >= max(os.path.getmtime(src), os.path.getmtime(hdr)):
        return so
    opt = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=all"] if sanitize else ["-O2"]
    cmd = ["g++"] + opt + ["-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-pthread", "-o", so, src]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return so


class GasDesc(C.Structure):
    _fields_ = [("n_bins", C.c_int32), ("e_max_eV", C.c_double), ("n_levels", C.c_int32),
                ("cum_rate", C.c_void_p), ("level_type", C.c_void_p), ("level_loss_eV", C.c_void_p),
                ("level_recoil", C.c_void_p), ("level_ob_w_eV", C.c_void_p), ("nu_hat", C.c_double),
                ("scat_xi", C.c_void_p), ("level_penning_prob", C.c_void_p), ("level_penning_eV", C.c_void_p),
                ("kT_eV", C.c_double)]


class SlabDesc(C.Structure):
    _fields_ = [("z_lo", C.c_double), ("z_hi", C.c_double), ("kind", C.c_int32), ("E", C.c_double * 3),
                ("nodes", C.c_void_p), ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("origin", C.c_double * 3), ("spacing", C.c_double * 3), ("bc_x", C.c_int32), ("bc_y", C.c_int32),
                ("period_x", C.c_double), ("period_y", C.c_double),
                ("n_mesh_nodes", C.c_int64), ("n_tets", C.c_int64), ("node_xyz", C.c_void_p), ("node_V", C.c_void_p),
                ("tet_nodes", C.c_void_p), ("tet_gas", C.c_void_p)]


class FieldDescC(C.Structure):
    _fields_ = [("slabs", C.POINTER(SlabDesc)), ("n_slabs", C.c_int32), ("B", C.c_double * 3),
                ("xy_lo", C.c_double * 2), ("xy_hi", C.c_double * 2)]


class SignalC(C.Structure):
    _fields_ = [("weighting", C.POINTER(FieldDescC)), ("t0", C.c_double), ("dt_bin", C.c_double), ("n_bins", C.c_int32),
                ("signal", C.c_void_p)]


class IonOpts(C.Structure):
    _fields_ = [("mobility_pos", C.c_double), ("mobility_neg", C.c_double), ("step_cm", C.c_double), ("t_max", C.c_double),
                ("max_steps", C.c_int32)]


class RunOpts(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("t_max", C.c_double), ("n_threads", C.c_int32), ("id_offset", C.c_uint64),
                ("flags", C.c_uint32), ("signal", C.POINTER(SignalC))]


BANDED = 1


class Outputs(C.Structure):
    _fields_ = [("capacity", C.c_int64), ("id", C.c_void_p), ("avalanche", C.c_void_p), ("status", C.c_void_p),
                ("n_steps", C.c_void_p), ("birth", C.c_void_p), ("end", C.c_void_p), ("per_avalanche", C.c_void_p),
                ("tallies_u64", C.c_void_p), ("tallies_f64", C.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.avmo_last_error.restype = C.c_char_p
        _lib.avmo_run.restype = C.c_int32
        _lib.avmo_step_batch.restype = C.c_int32
        _lib.avmo_field_eval.restype = C.c_int32
        _lib.avmo_majorant.restype = C.c_int32
        _lib.avmo_ion_drift.restype = C.c_int32
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


class _Keep:
    """Holds the numpy arrays a C descriptor points into."""

    def __init__(self):
        self.refs = []


def gas_desc(gas) -> tuple:
    k = _Keep()
    cum = np.ascontiguousarray(gas.cum_rate, dtype=np.float64)
    ty = np.ascontiguousarray(gas.level_type, dtype=np.uint8)
    lo = np.ascontiguousarray(gas.level_loss, dtype=np.float64)
    rc = np.ascontiguousarray(gas.level_recoil, dtype=np.float64)
    w = np.ascontiguousarray(gas.level_ob_w, dtype=np.float64)
    k.refs += [cum, ty, lo, rc, w]
    opt = []
    for name in ("scat_xi", "level_penning_prob", "level_penning_eV"):      # NEXT-3 extensions: optional
        a = getattr(gas, name, None)
        if a is None:
            opt.append(None)
        else:
            a = np.ascontiguousarray(a, dtype=np.float64)
            k.refs.append(a)
            opt.append(_p(a).value)
    d = GasDesc(int(gas.n_bins), float(gas.e_max), int(cum.shape[1]), _p(cum).value, _p(ty).value, _p(lo).value,
                _p(rc).value, _p(w).value, float(gas.nu_hat), opt[0], opt[1], opt[2], float(getattr(gas, "kT_eV", 0.0)))
    return d, k


def field_desc(field) -> tuple:
    k = _Keep()
    n = len(field.slabs)
    arr = (SlabDesc * n)()
    for i, s in enumerate(field.slabs):
        a = arr[i]
        a.z_lo, a.z_hi, a.kind = s.z_lo, s.z_hi, s.kind
        a.E[:] = s.E
        if s.nodes is not None:
            nodes = np.ascontiguousarray(s.nodes, dtype=np.float32)
            k.refs.append(nodes)
            a.nodes = _p(nodes).value
            a.nz, a.ny, a.nx = nodes.shape[:3]
        a.origin[:] = s.origin
        a.spacing[:] = s.spacing
        a.bc_x, a.bc_y, a.period_x, a.period_y = s.bc_x, s.bc_y, s.period_x, s.period_y
        m = getattr(s, "mesh", None)
        if m is not None:                       # kind 2: unstructured tetrahedral map (NEXT-2)
            xyz = np.ascontiguousarray(m.node_xyz, dtype=np.float64); v = np.ascontiguousarray(m.node_V, dtype=np.float64)
            tn = np.ascontiguousarray(m.tet_nodes, dtype=np.int32); tg = np.ascontiguousarray(m.tet_gas, dtype=np.uint8)
            k.refs += [xyz, v, tn, tg]
            a.n_mesh_nodes, a.n_tets = xyz.shape[0], tn.shape[0]
            a.node_xyz, a.node_V, a.tet_nodes, a.tet_gas = _p(xyz).value, _p(v).value, _p(tn).value, _p(tg).value
    k.refs.append(arr)
    d = FieldDescC(arr, n, (C.c_double * 3)(*field.B), (C.c_double * 2)(*field.xy_lo), (C.c_double * 2)(*field.xy_hi))
    return d, k


def philox(seed, ident, n, block) -> np.ndarray:
    out = (C.c_uint32 * 4)()
    lib().avmo_philox(C.c_uint64(seed), C.c_uint64(ident), C.c_uint32(n), C.c_uint32(block), out)
    return np.array(out[:], dtype=np.uint32)


def uniform_pair(seed, ident, n, block):
    out = (C.c_double * 2)()
    lib().avmo_uniform_pair(C.c_uint64(seed), C.c_uint64(ident), C.c_uint32(n), C.c_uint32(block), out)
    return out[0], out[1]


def field_eval(field, r):
    """r: [3, n] -> E [3, n], mask [n], slab [n]."""
    r = np.ascontiguousarray(r, dtype=np.float64)
    n = r.shape[1]
    E = np.zeros((3, n)); m = np.zeros(n); sl = np.zeros(n, dtype=np.int32)
    fd, _k = field_desc(field)
    rc = lib().avmo_field_eval(C.byref(fd), C.c_int64(n), _p(r), _p(E), _p(m), _p(sl))
    if rc != 0:
        raise RuntimeError(lib().avmo_last_error().decode())
    return E, m, sl


@dataclass
class StepResult:
    state: np.ndarray      # [8, n]
    event: np.ndarray
    status: np.ndarray
    bin: np.ndarray
    child: np.ndarray      # [8, n]
    child_id: np.ndarray


def majorant(gas):
    """The banded-rate table of this gas: (a2 [J], nu [K, J+1], dtmax [K, J+1], shift)."""
    gd, _kg = gas_desc(gas)
    shp = (C.c_int32 * 3)()
    assert lib().avmo_majorant(C.byref(gd), shp, None, None, None) == 0
    K, J, shift = shp[0], shp[1], shp[2]
    a2 = np.zeros(J); nu = np.zeros((K, J + 1)); dt = np.zeros((K, J + 1))
    assert lib().avmo_majorant(C.byref(gd), shp, _p(a2), _p(nu), _p(dt)) == 0
    return a2, nu, dt, shift


def step_batch(gas, field, seed, state, ids, n_idx, t_max=float("inf"), flags=0) -> StepResult:
    state = np.ascontiguousarray(state, dtype=np.float64)
    n = state.shape[1]
    ids = np.ascontiguousarray(ids, dtype=np.uint64)
    n_idx = np.ascontiguousarray(n_idx, dtype=np.uint32)
    out = np.zeros((8, n)); ev = np.zeros(n, dtype=np.int32); st = np.zeros(n, dtype=np.int32)
    bn = np.zeros(n, dtype=np.int32); ch = np.zeros((8, n)); cid = np.zeros(n, dtype=np.uint64)
    gd, _kg = gas_desc(gas)
    fd, _kf = field_desc(field)
    rc = lib().avmo_step_batch(C.byref(gd), C.byref(fd), C.c_uint64(seed), C.c_double(t_max), C.c_int64(n), _p(state),
                               _p(ids), _p(n_idx), _p(out), _p(ev), _p(st), _p(bn), _p(ch), _p(cid), C.c_uint32(flags))
    if rc != 0:
        raise RuntimeError(lib().avmo_last_error().decode())
    return StepResult(out, ev, st, bn, ch, cid)


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
    n_rate_violations: int = 0  # banded runs: steps whose bin's total rate exceeded the band's rate (always 0)
    signal: np.ndarray = None   # induced charge per time bin [e] when a signal description was given

    def sorted_by_id(self):
        o = np.argsort(self.id, kind="stable")
        return RunResult(self.n, self.id[o], self.avalanche[o], self.status[o], self.n_steps[o], self.birth[:, o],
                         self.end[:, o], self.per_avalanche, self.tallies_u64, self.tallies_f64, self.rc,
                         self.n_rate_violations, self.signal)


def _signal_c(weighting, t0, dt_bin, signal):
    wd, kw = field_desc(weighting)
    s = SignalC(C.pointer(wd), float(t0), float(dt_bin), int(signal.shape[0]), _p(signal).value)
    return s, (wd, kw)


def run(gas, field, primaries, seed=0, t_max=float("inf"), capacity=None, n_threads=1, allow_overflow=False,
        id_offset=0, flags=0, signal=None) -> RunResult:
    """signal: None or (weighting FieldDesc, t0, dt_bin, n_bins) — the induced charge per time bin is returned in
    RunResult.signal (NEXT-4)."""
    prim = np.ascontiguousarray(primaries, dtype=np.float64)
    np_ = prim.shape[0]
    cap = int(capacity if capacity is not None else max(4 * np_, 1 << 16))
    L = gas.n_levels
    ident = np.zeros(cap, dtype=np.uint64); av = np.zeros(cap, dtype=np.uint32); st = np.zeros(cap, dtype=np.int32)
    ns = np.zeros(cap, dtype=np.uint32); birth = np.zeros((5, cap)); end = np.zeros((8, cap))
    pa = np.zeros((max(np_, 1), 3), dtype=np.uint64); tu = np.zeros(L + 6, dtype=np.uint64); tf = np.zeros(5)
    gd, _kg = gas_desc(gas)
    fd, _kf = field_desc(field)
    o = Outputs(cap, _p(ident), _p(av), _p(st), _p(ns), _p(birth), _p(end), _p(pa), _p(tu), _p(tf))
    sig_arr, sig_c, _ks = None, None, None
    if signal is not None:
        sig_arr = np.zeros(int(signal[3]))
        sig_c, _ks = _signal_c(signal[0], signal[1], signal[2], sig_arr)
    opts = RunOpts(int(seed), float(t_max), int(n_threads), int(id_offset), int(flags), C.pointer(sig_c) if sig_c is not None else None)
    n_out = C.c_int64(0)
    rc = lib().avmo_run(C.byref(gd), C.byref(fd), _p(prim), C.c_int64(np_), C.byref(opts), C.byref(o), C.byref(n_out))
    if rc == -2 and not allow_overflow:
        raise MemoryError("oracle: capacity exceeded")
    if rc not in (0, -2):
        raise RuntimeError(lib().avmo_last_error().decode())
    n = n_out.value
    return RunResult(n, ident[:n], av[:n], st[:n], ns[:n], birth[:, :n], end[:, :n], pa[:np_], tu[:L + 5], tf, rc, int(tu[L + 5]), sig_arr)


@dataclass
class IonResult:
    end: np.ndarray        # [4, 2n]: x, y, z, t; entry s = positive ion born with electron s, n + s = negative ion of electron s
    status: np.ndarray     # [2n]; -1 = no such ion
    n_steps: np.ndarray
    signal: np.ndarray = None


def ion_drift(field, run_result, n_primaries, mobility_pos, mobility_neg, step_cm, t_max=float("inf"), max_steps=1 << 20,
              signal=None) -> IonResult:
    r = run_result
    n = int(r.n)
    birth = np.ascontiguousarray(r.birth, dtype=np.float64); end = np.ascontiguousarray(r.end, dtype=np.float64)
    status = np.ascontiguousarray(r.status, dtype=np.int32)
    ie = np.zeros((4, 2 * n)); ist = np.zeros(2 * n, dtype=np.int32); ins = np.zeros(2 * n, dtype=np.uint32)
    fd, _kf = field_desc(field)
    sig_arr, sig_c, _ks = None, None, None
    if signal is not None:
        sig_arr = np.zeros(int(signal[3]))
        sig_c, _ks = _signal_c(signal[0], signal[1], signal[2], sig_arr)
    io = IonOpts(float(mobility_pos), float(mobility_neg), float(step_cm), float(t_max), int(max_steps))
    rc = lib().avmo_ion_drift(C.byref(fd), C.byref(sig_c) if sig_c is not None else None, C.byref(io), C.c_int64(n), C.c_int64(n_primaries),
                              C.c_int64(birth.shape[1]), _p(birth), C.c_int64(end.shape[1]), _p(end), _p(status), _p(ie), _p(ist), _p(ins))
    if rc != 0:
        raise RuntimeError(lib().avmo_last_error().decode())
    return IonResult(ie, ist, ins, sig_arr)
