"""Scenarios run by tests/test_oracle_sanitizers.py in a subprocess whose oracle is the ASan + UBSan build
(AVMO_SANITIZED=1, libasan preloaded).  Each exercises tables the oracle indexes: the band table of the energy-banded
rate, the bucket grid and element records of a tetrahedral map, a grid map with folds, the signal bins and the ion arrays,
the capacity limit.  Results are checked only for being complete; the sanitizers do the checking."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from oracle import avmo                                            # noqa: E402
from paper_2509_15377_b200.gen import fields, gas, primaries, tetmesh   # noqa: E402

assert avmo._SO.endswith("libavmo_san.so"), avmo._SO
avmo.build()
g0 = gas.gas_g0()
H = 2e-4

# 1. banded run, uniform field with B (band table, cut flights, helix), several threads
fd = fields.uniform_gap((0.0, 0.0, -30000.0), 0.0, 50e-4, (0.2, 0.1, 0.5))
p = primaries.isotropic_primaries(150, 1)
for flags in (0, 1):
    r = avmo.run(g0, fd, p, seed=1, n_threads=3, flags=flags)
    assert r.n >= 150 and np.all(r.status >= 1)
# capacity limit: children that do not fit are dropped, nothing is written beyond the arrays
try:
    avmo.run(g0, fields.uniform_gap((0.0, 0.0, -60000.0), 0.0, 100e-4), p, seed=1, capacity=400, n_threads=2)
except Exception as e:                                             # the wrapper reports the overflow
    print("capacity:", str(e)[:80])

# 2. tetrahedral map with solid and removed elements: field evaluation (vertices, outside points, folds) and a run with signal
V = lambda x, y, z: -3000.0 * z - 30.0 * np.tanh((z - 20e-4) / 5e-4) * (1.5 - np.exp(-(x * x + y * y) / (8e-4) ** 2))
foil = lambda x, y, z: (np.abs(z - 20e-4) < 4e-4) & (x * x + y * y > (8e-4) ** 2)
metal = lambda x, y, z: (np.abs(z - 20e-4) < 1.5e-4) & (x * x + y * y > (12e-4) ** 2)
mesh = tetmesh.kuhn_mesh(9, 9, 21, (H, H, H), V, seed=2, solid=foil, removed=metal)
Lx, Lz = 8 * H, 20 * H
ft = fields.FieldDesc([fields.tet_slab(mesh, (0.0, 0.0, 0.0), 0.0, Lz, fields.BC_MIRROR, fields.BC_PERIODIC, Lx, Lx),
                       fields.Slab(Lz, Lz + 10e-4, fields.KIND_UNIFORM, (0.0, 0.0, 3000.0))])
rng = np.random.default_rng(0)
r3 = rng.uniform(-1, 1, size=(3, 20000)) * np.array([5 * Lx, 5 * Lx, 0.0])[:, None]
r3[2] = rng.uniform(-5e-4, Lz + 15e-4, 20000)
r3[:, :300] = mesh.node_xyz[mesh.tet_nodes[:300, 0]].T
r3[:, 300] = np.nan
E, m, sl = avmo.field_eval(ft, r3)
assert (sl == -1).sum() > 100 and (m == 0).sum() > 100
wf = fields.uniform_gap((0.0, 0.0, 1.0 / (Lz + 10e-4)), 0.0, Lz + 10e-4)
pt = primaries.isotropic_primaries(60, 4, pos=(0.0, 0.0, Lz + 5e-4), xy_box=((0.0, Lx), (0.0, Lx)))
for flags in (0, 1):
    rt = avmo.run(g0, ft, pt, seed=4, n_threads=2, flags=flags, t_max=40.0, signal=(wf, 0.0, 0.05, 50))
    assert rt.n >= 60 and rt.signal.shape == (50,)
# 3. ion drift through the mesh, with a signal whose bins the late ions overrun
ions = avmo.ion_drift(ft, rt, 60, 1.5e-9, 2.0e-9, 0.5e-4, t_max=3e4, signal=(wf, 0.0, 100.0, 20))
assert ions.status.shape[0] == 2 * rt.n

# 4. grid map with mirror / periodic folds and material, steps from states at and beyond the edges
nodes = (rng.normal(size=(12, 9, 7, 4)) * 2e4).astype(np.float32)
nodes[..., 2] -= 3e4
nodes[..., 3] = (rng.uniform(size=(12, 9, 7)) > 0.1).astype(np.float32)
fm = fields.FieldDesc([fields.grid_slab(nodes, (0, 0, 0), (1e-4, 1e-4, 1e-4), 0.0, 11e-4, fields.BC_MIRROR, fields.BC_PERIODIC, 6e-4, 8e-4)])
n = 4000
st = np.zeros((8, n)); st[0:2] = rng.uniform(-30e-4, 30e-4, size=(2, n)); st[2] = rng.uniform(-1e-4, 12e-4, n)
k = rng.normal(size=(3, n)); st[5:8] = k / np.linalg.norm(k, axis=0); st[4] = np.exp(rng.uniform(np.log(0.01), np.log(60.0), n))
ids = rng.integers(0, 2 ** 64, n, dtype=np.uint64); nidx = rng.integers(0, 1 << 24, n, dtype=np.uint64).astype(np.uint32)
for flags in (0, 1):
    sb = avmo.step_batch(g0, fm, 3, st, ids, nidx, flags=flags)
    assert sb.event.shape[0] == n
# 5. NEXT-3 extensions: anisotropic table, Penning, thermal gas
gx = gas.gas_g0(n_bins=2000)
gx.scat_xi = rng.uniform(-0.9, 0.9, size=gx.cum_rate.shape)
gx.level_penning_prob = np.where(np.asarray(gx.level_type) == 1, 0.3, 0.0)
gx.level_penning_eV = np.full(len(gx.level_type), 2.0)
gx.kT_eV = 0.02526
rx = avmo.run(gx, fields.uniform_gap((0.0, 0.0, -30000.0), 0.0, 50e-4), primaries.isotropic_primaries(100, 9), seed=9, n_threads=2)
assert rx.n >= 100
print("sanitized oracle scenarios: ok")
