"""Pin C17: an independent transcription of one transport step S0-S9 in 40-digit arithmetic.

Written from the S0-S9 table and readings R1-R20 of SURVEY.md §8(c) (restated in DESIGN.md §3), in their order and
notation, with mpmath reals and Python integers.  It calls nothing under oracle/ and nothing under
paper_2509_15377_b200/csrc/; it reads the plain-data inputs (GasTable, FieldDesc) only.  Its own Philox is the
published algorithm (Salmon et al., SC'11) on Python ints — a fourth implementation beside the oracle's, the
generators' and the device's.  Used by tests/test_oracle_pins_composition.py; slow by design (pure Python).
"""
from mpmath import mp, mpf

mp.dps = 40

C2 = mpf("0.05930969584745753")
INV_C2SQ = mpf("284.28150518042008")
KAPPA = mpf("0.0017588200107589609")
OMEGA1 = mpf("175.88200107589608")
EPS_FLOOR = mpf("1e-10")
M32 = 0xFFFFFFFF
STEP_LIMIT = 0xFFFFFFF0


def philox(seed, ident, n, block):
    c = [n & M32, block & M32, ident & M32, (ident >> 32) & M32]
    k0, k1 = seed & M32, (seed >> 32) & M32
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k0, p1 & M32, (p0 >> 32) ^ c[3] ^ k1, p0 & M32]
        k0, k1 = (k0 + 0x9E3779B9) & M32, (k1 + 0xBB67AE85) & M32
    return c


def uniforms(seed, ident, n, block):
    w = philox(seed, ident, n, block)
    two52 = mpf(2) ** -52
    return ((((w[0] << 32) | w[1]) >> 12) + mpf("0.5")) * two52, ((((w[2] << 32) | w[3]) >> 12) + mpf("0.5")) * two52


def _fold(x, origin, h, n, bc, P):
    """R15.  Returns (q, flip) or None when outside a bc-none grid."""
    q = x - origin
    if bc == 0:
        return (q, False) if 0 <= q <= (n - 1) * h else None
    if bc == 1:
        return q - P * mp.floor(q / P), False
    q = q - 2 * P * mp.floor(q / (2 * P))
    return (2 * P - q, True) if q > P else (q, False)


def _cell(q, h, n):
    s = q / h
    i = max(min(int(mp.floor(s)), n - 2), 0)
    return i, s - i


def field_at(fd, x, y, z):
    """S0 / R14 / R15.  Returns (E[3], mask) or -status."""
    S = fd.slabs
    if z < S[0].z_lo:
        return -1
    if z > S[-1].z_hi:
        return -2
    if x < fd.xy_lo[0] or x > fd.xy_hi[0] or y < fd.xy_lo[1] or y > fd.xy_hi[1]:
        return -3
    s = S[-1]
    for cand in S:
        if z < cand.z_hi:
            s = cand
            break
    if s.kind == 0:
        return [mpf(v) for v in s.E], mpf(1)
    nz, ny, nx, _ = s.nodes.shape
    fx = _fold(x, mpf(s.origin[0]), mpf(s.spacing[0]), nx, s.bc_x, mpf(s.period_x))
    fy = _fold(y, mpf(s.origin[1]), mpf(s.spacing[1]), ny, s.bc_y, mpf(s.period_y))
    if fx is None or fy is None:
        return -3
    i, wx = _cell(fx[0], mpf(s.spacing[0]), nx)
    j, wy = _cell(fy[0], mpf(s.spacing[1]), ny)
    k, wz = _cell(z - mpf(s.origin[2]), mpf(s.spacing[2]), nz)
    out = []
    for c in range(4):
        N = lambda kk, jj, ii: mpf(float(s.nodes[kk, jj, ii, c]))
        c00 = N(k, j, i) + wx * (N(k, j, i + 1) - N(k, j, i))
        c10 = N(k, j + 1, i) + wx * (N(k, j + 1, i + 1) - N(k, j + 1, i))
        c01 = N(k + 1, j, i) + wx * (N(k + 1, j, i + 1) - N(k + 1, j, i))
        c11 = N(k + 1, j + 1, i) + wx * (N(k + 1, j + 1, i + 1) - N(k + 1, j + 1, i))
        c0 = c00 + wy * (c10 - c00)
        c1 = c01 + wy * (c11 - c01)
        out.append(c0 + wz * (c1 - c0))
    return [-out[0] if fx[1] else out[0], -out[1] if fy[1] else out[1], out[2]], out[3]


def _cross(a, b):
    return [a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]]


def _dot(a, b):
    return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]


def step(gas, fd, seed, t_max, state, ident, n):
    """One step from state = (x, y, z, t, eps, kx, ky, kz) (floats).  Returns a dict with the oracle's step outputs:
    state (8 mpf), event (-2 ended before the decision, -1 null, else level), status, bin, child (8 mpf or None), child_id."""
    r = [mpf(state[0]), mpf(state[1]), mpf(state[2])]
    t, eps = mpf(state[3]), mpf(state[4])
    k = [mpf(state[5]), mpf(state[6]), mpf(state[7])]
    out = {"event": -2, "status": 0, "bin": -1, "child": None, "child_id": 0}
    f0 = field_at(fd, *r)                                                    # S0
    assert not isinstance(f0, int), "step() starts in the domain"
    E, _ = f0
    n_s = n                                                                  # S1
    u1, u2 = uniforms(seed, ident, n_s, 0)
    nu_hat = mpf(gas.resolved_nu_hat())
    dt = -mp.log(u1) * (1 / nu_hat)                                          # S2
    v0 = [C2 * mp.sqrt(eps) * ki for ki in k]                                # S3
    a = [-KAPPA * Ei for Ei in E]
    B = [mpf(b) for b in fd.B]
    Bn2 = _dot(B, B)
    if Bn2 == 0:
        r1 = [r[i] + v0[i] * dt + a[i] * dt * dt / 2 for i in range(3)]
        v1 = [v0[i] + a[i] * dt for i in range(3)]
    else:
        Bn = mp.sqrt(Bn2)
        bh = [b / Bn for b in B]
        omega = OMEGA1 * Bn
        apar = [_dot(a, bh) * b for b in bh]
        vd = [mpf("1e-5") * c / Bn2 for c in _cross(E, B)]
        vpar = [_dot(v0, bh) * b for b in bh]
        w0 = [v0[i] - vpar[i] - vd[i] for i in range(3)]
        bxw = _cross(bh, w0)
        th = omega * dt
        v1 = [vpar[i] + apar[i] * dt + vd[i] + w0[i] * mp.cos(th) + bxw[i] * mp.sin(th) for i in range(3)]
        r1 = [r[i] + vpar[i] * dt + apar[i] * dt * dt / 2 + vd[i] * dt
              + (w0[i] * mp.sin(th) + bxw[i] * 2 * mp.sin(th / 2) ** 2) / omega for i in range(3)]
    s = _dot(v1, v1)                                                         # S4
    e1 = max(s * INV_C2SQ, EPS_FLOOR)
    k1 = [vi / mp.sqrt(s) for vi in v1] if s > 0 else k
    t1 = t + dt
    n1 = n_s + 1
    out["state"] = r1 + [t1, e1] + k1
    out["n"] = n1
    f1 = field_at(fd, *r1)                                                   # S5
    if isinstance(f1, int):
        out["status"] = -f1
        return out
    if f1[1] < mpf("0.5"):
        out["status"] = 4
        return out
    if t1 > t_max:
        out["status"] = 6
        return out
    if n1 >= STEP_LIMIT:
        out["status"] = 7
        return out
    nb, L = gas.n_bins, gas.n_levels                                         # S6
    b = min(nb - 1, int(mp.floor(e1 * (mpf(nb) / mpf(gas.e_max)))))
    out["bin"] = b
    row = [mpf(float(c)) for c in gas.cum_rate[b]]
    x = u2 * nu_hat                                                          # S7
    if x >= row[L - 1]:
        out["event"] = -1
        return out
    lvl = next(l for l in range(L) if row[l] > x)                            # S8
    out["event"] = lvl
    ty = int(gas.level_type[lvl])
    if ty == 3:                                                              # S9a
        out["status"] = 5
        return out
    u3, u4 = uniforms(seed, ident, n_s, 1)                                   # S9b
    ct = 1 - 2 * u3
    st = 2 * mp.sqrt(u3 * (1 - u3))
    phi = 2 * mp.pi * u4
    if ty == 0:                                                              # S9c
        e2 = e1 * (1 - mpf(float(gas.level_recoil[lvl])) * (1 - ct))
    elif ty == 1:
        e2 = max(e1 - mpf(float(gas.level_loss[lvl])), EPS_FLOOR)
    else:
        u5, u6 = uniforms(seed, ident, n_s, 2)
        u7, _ = uniforms(seed, ident, n_s, 3)
        ea = max(e1 - mpf(float(gas.level_loss[lvl])), mpf(0))
        w = mpf(float(gas.level_ob_w[lvl]))
        es = w * mp.tan(u5 * mp.atan(ea / (2 * w)))
        e2 = max(ea - es, EPS_FLOOR)
        sc = 2 * mp.sqrt(u6 * (1 - u6))
        out["child"] = r1 + [t1, max(es, EPS_FLOOR), sc * mp.cos(2 * mp.pi * u7), sc * mp.sin(2 * mp.pi * u7), 1 - 2 * u6]
        wd = philox(seed, ident, n_s, 0xFFFFFFFF)
        out["child_id"] = wd[0] + (wd[1] << 32)
    sg = mpf(1) if k1[2] >= 0 else mpf(-1)                                   # S9d (Duff et al. 2017); copysign(1, +0) = 1
    A = -1 / (sg + k1[2])
    Bq = k1[0] * k1[1] * A
    b1 = [1 + sg * k1[0] * k1[0] * A, sg * Bq, -sg * k1[0]]
    b2 = [Bq, sg + k1[1] * k1[1] * A, -k1[1]]
    k2 = [ct * k1[i] + st * (mp.cos(phi) * b1[i] + mp.sin(phi) * b2[i]) for i in range(3)]
    nk = mp.sqrt(_dot(k2, k2))
    out["state"] = r1 + [t1, e2] + [c / nk for c in k2]
    return out
