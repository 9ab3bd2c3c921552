"""Pins for Algorithm 1 steps 7-14 and Algorithm 2: LHCS, RK4,
reconstruction, D / B layout.  P12 of DESIGN.md: these parts are PARITY UNPINNED against the
authors' implementation (no vector in the paper); what is checked here is the mathematics -- Eq. (1)
hand-evaluated, RK4 against a high-accuracy ODE solve, IEEE field invariants, hand-worked
reconstructions -- and the BITS of the readings this repository fixed: a pure-Python binary64
restatement of SURVEY.md 8(c) steps 2-7 and 10 (py_* below: Python floats and ints only, no numpy
arithmetic, no call into the oracle) must reproduce the oracle's RK4 states, whitening, IR records, D
and B bit for bit, and both must reproduce the frozen vector tests/golden/derive_tiny.txt.
"""
import os
import struct
import tempfile

import numpy as np
import pytest

from conftest import read_golden

KEY = (3.141592653589793, 2.718281828459045, 1.4142135623730951, 1.7320508075688772)


@pytest.mark.parametrize("row", read_golden("lhcs_eq1_worked.txt"))
def test_rhs_hand_evaluated(orc, row):
    v = [float(x) for x in row]
    got = orc.lhcs_rhs(v[:4], v[4])
    assert got.tolist() == v[5:9]


def test_rhs_divergence_and_symmetry(orc):
    """Eq. (1): trace of the Jacobian = -(sigma + 1 + beta) + gamma everywhere; the system is
    invariant under (x, y, w) -> (-x, -y, -w), z fixed."""
    rng = np.random.default_rng(0)
    for _ in range(20):
        s = rng.uniform(-20, 20, 4)
        g = float(rng.uniform(-1.52, -0.06))
        eps = 1e-6
        div = 0.0
        for k in range(4):
            e = np.zeros(4); e[k] = eps
            div += (orc.lhcs_rhs(s + e, g)[k] - orc.lhcs_rhs(s - e, g)[k]) / (2 * eps)
        assert abs(div - (-(10 + 1 + 8 / 3) + g)) < 1e-6
        f = orc.lhcs_rhs(s, g)
        fm = orc.lhcs_rhs(s * np.array([-1, -1, 1, -1]), g)
        assert np.allclose(fm, f * np.array([-1, -1, 1, -1]), rtol=0, atol=1e-12)


def test_rk4_matches_high_accuracy_ode_solve(orc):
    """One oracle step (dt = 0.005) against scipy's DOP853 at rtol 1e-13.  Measured: the local
    error of the oracle's RK4 is <= 3.4e-6 on these states; Euler is off by 2e-2, midpoint RK2 by
    5e-4, a dropped factor 2 on k3 by 1e-1, a wrong sign in Eq. (1) by more.  (RK3 vs RK4 is
    separated by test_rk4_order_four.)"""
    from scipy.integrate import solve_ivp

    def f(t, s, g):
        x, y, z, w = s
        return [10 * (y - x) + w, 28 * x - y - x * z, x * y - 8 / 3 * z, -y * z + g * w]

    rng = np.random.default_rng(1)
    for _ in range(10):
        s = rng.uniform(-15, 15, 4)
        g = float(rng.uniform(-1.52, -0.06))
        ref = solve_ivp(f, (0, 0.005), s, args=(g,), method="DOP853", rtol=1e-13, atol=1e-13).y[:, -1]
        got = orc.rk4(s, g, 1)
        assert np.max(np.abs(got - ref)) < 2e-5
        # 40 steps = t 0.2: global error O(dt^4), still far below what a wrong scheme gives
        ref = solve_ivp(f, (0, 0.2), s, args=(g,), method="DOP853", rtol=1e-13, atol=1e-13).y[:, -1]
        assert np.max(np.abs(orc.rk4(s, g, 40) - ref)) < 2e-3


def test_rk4_order_four(orc):
    """Convergence order: the error against the ODE solve over t = 0.005 (1 oracle step) is
    ~32x (2^5) the per-step error class; checked through the step-doubling estimate
    |y_1step(2dt-equivalent)| -- here: oracle's fixed-dt trajectory over 2 steps vs 1 step of
    an independent plain RK4 with dt = 0.01 differs by ~ (2^4 - 1)/2^4 of the coarse error."""
    from scipy.integrate import solve_ivp

    def f(t, s, g=-1.0):
        x, y, z, w = s
        return np.array([10 * (y - x) + w, 28 * x - y - x * z, x * y - 8 / 3 * z, -y * z + g * w])

    s = np.array([5.0, -7.0, 20.0, 3.0])
    T = 0.02  # 4 oracle steps
    ref = solve_ivp(f, (0, T), s, method="DOP853", rtol=1e-13, atol=1e-14).y[:, -1]
    err_fine = np.max(np.abs(orc.rk4(s, -1.0, 4) - ref))

    def rk4(s, dt):  # textbook RK4, only used at the coarse step to measure the ratio
        k1 = f(0, s); k2 = f(0, s + dt / 2 * k1); k3 = f(0, s + dt / 2 * k2); k4 = f(0, s + dt * k3)
        return s + dt / 6 * (k1 + 2 * k2 + 2 * k3 + k4)

    c = s.copy()
    for _ in range(2):
        c = rk4(c, 0.01)
    err_coarse = np.max(np.abs(c - ref))
    assert 8 < err_coarse / err_fine < 32  # ~16 for a 4th-order scheme


def test_trajectories_bounded_and_chaotic(orc):
    """LHCS is hyper-chaotic for -1.52 <= gamma <= -0.06: states stay bounded and
    a 1e-14 perturbation grows to O(1) (the basis of Fig. 6)."""
    for g in (-1.52, -1.0, -0.06):
        s = orc.rk4(KEY, g, 20000)
        assert np.all(np.isfinite(s)) and np.max(np.abs(s)) < 400
    a = orc.rk4(KEY, -1.0, 20000)
    b = orc.rk4((KEY[0] + 1e-14,) + KEY[1:], -1.0, 20000)
    assert np.max(np.abs(a - b)) > 1e-2


@pytest.mark.parametrize("row", read_golden("reconstruct_worked.txt"))
def test_reconstruct_hand_worked(orc, row):
    v, hb, want = float(row[0]), bytes.fromhex(row[1]), float(row[2])
    assert orc.reconstruct(v, hb) == want


def test_reconstruct_ieee_invariants(orc):
    """Result in [0, u+1); only mantissa bits 0..47 of the fraction change; integer part follows
    the XOR/mod rule; two reconstructions with hashes differing in one byte differ."""
    rng = np.random.default_rng(5)
    for _ in range(2000):
        v = float(rng.uniform(-300, 300))
        hb = rng.integers(0, 256, 8, dtype=np.uint8).tobytes()
        r = orc.reconstruct(v, hb)
        assert 0.0 <= r < 41.0
        a = abs(v)
        ip = int(a)
        fr = a - ip
        want_I = ((ip & 0xFFFF) ^ (hb[0] | hb[1] << 8)) % 40
        bits = struct.unpack("<Q", struct.pack("<d", fr))[0] ^ int.from_bytes(hb[2:8], "little")
        frac = struct.unpack("<d", struct.pack("<Q", bits))[0]
        assert 0.0 <= frac < 1.0
        assert (bits >> 48) == (struct.unpack("<Q", struct.pack("<d", fr))[0] >> 48)
        assert r == want_I + frac
        # a flipped bit of hb0/hb1 always changes the integer part (2^k mod 40 != 0); low fraction
        # bits may be absorbed by the rounding of the final add, so they are not asserted on
        hb2 = bytearray(hb); hb2[int(rng.integers(2))] ^= 1 << int(rng.integers(8))
        assert orc.reconstruct(v, bytes(hb2)) != r


# ---------------------------------------------------------------------------------------------------
# Pure-Python binary64 restatement of SURVEY.md 8(c) (PAPER.md:35-43 Eq. 1, :55, :59).  CPython floats are
# IEEE binary64, every operator below is one correctly rounded operation and nothing can be contracted
# into an FMA, so the expression order written here IS the arithmetic.  Nothing below calls the oracle.
# ---------------------------------------------------------------------------------------------------
DT = 0.005
HALF_DT = 0.5 * DT
DT_6 = DT / 6.0
BETA = 8.0 / 3.0
K_M, N0, U = 16, 20000, 40


def py_f(x, y, z, w, g):
    """Step 10: f = (10 (y - x) + w, (28 x - y) - x z, x y - (8/3) z, (-(y z)) + gamma w)."""
    return (10.0 * (y - x) + w, (28.0 * x - y) - x * z, x * y - BETA * z, (-(y * z)) + g * w)


def py_rk4_step(s, g):
    """Step 10: k1 = f(s), k2 = f(s + (dt/2) k1), k3 = f(s + (dt/2) k2), k4 = f(s + dt k3),
    s' = s + (dt/6) (((k1 + 2 k2) + 2 k3) + k4)."""
    k1 = py_f(s[0], s[1], s[2], s[3], g)
    k2 = py_f(s[0] + HALF_DT * k1[0], s[1] + HALF_DT * k1[1], s[2] + HALF_DT * k1[2], s[3] + HALF_DT * k1[3], g)
    k3 = py_f(s[0] + HALF_DT * k2[0], s[1] + HALF_DT * k2[1], s[2] + HALF_DT * k2[2], s[3] + HALF_DT * k2[3], g)
    k4 = py_f(s[0] + DT * k3[0], s[1] + DT * k3[1], s[2] + DT * k3[2], s[3] + DT * k3[3], g)
    return tuple(s[i] + DT_6 * (((k1[i] + 2.0 * k2[i]) + 2.0 * k3[i]) + k4[i]) for i in range(4))


def py_rk4(s, g, steps):
    s = tuple(float(v) for v in s)
    for _ in range(steps):
        s = py_rk4_step(s, g)
    return s


def py_reconstruct(v, hb):
    """Step 3: a = |v|, ip = floor(a), fr = a - ip; I = ((ip & 0xFFFF) ^ (hb0 | hb1 << 8)) mod u;
    the IEEE pattern of fr XOR the 48-bit little-endian integer hb2..hb7; v' = I + that double."""
    a = abs(v)
    ip = int(a)  # truncation = floor for a >= 0
    fr = a - float(ip)
    integer = ((ip & 0xFFFF) ^ (hb[0] | hb[1] << 8)) % U
    bits = struct.unpack("<Q", struct.pack("<d", fr))[0] ^ int.from_bytes(hb[2:8], "little")
    return float(integer) + struct.unpack("<d", struct.pack("<Q", bits))[0]


def _bits(vals):
    return struct.pack("<%dd" % len(vals), *[float(v) for v in vals])


def test_rk4_bits_match_pure_python_restatement(orc):
    """The 48 low mantissa bits of every iterate ARE the keystream: the oracle's RK4 must be the
    operation sequence of step 10 bit for bit -- 24 random states and gammas x 1500 steps, compared after every
    step for the first 50 and at the end.  A re-associated final sum, a fused multiply-add, dt/6 computed as
    dt * (1/6), or 8/3 written as 2.6666666666666665 +- 1 ulp all fail here."""
    rng = np.random.default_rng(2024)
    for _ in range(24):
        s = tuple(float(v) for v in rng.uniform(-25, 25, 4))
        g = float(rng.uniform(-1.52, -0.06))
        o, p = np.array(s), s
        for _k in range(50):
            o, p = orc.rk4(o, g, 1), py_rk4_step(p, g)
            assert _bits(o) == _bits(p)
        assert _bits(orc.rk4(s, g, 1500)) == _bits(py_rk4(s, g, 1500))


def test_single_rhs_and_constants_bits(orc):
    """Eq. 1's right-hand side alone, bit for bit, and the three rounded constants of step 10."""
    assert DT_6 == 0.005 / 6.0 and HALF_DT == 0.0025 and struct.pack(">d", BETA).hex() == "4005555555555555"
    rng = np.random.default_rng(7)
    for _ in range(200):
        s = [float(v) for v in rng.uniform(-60, 60, 4)]
        g = float(rng.uniform(-1.52, -0.06))
        assert _bits(orc.lhcs_rhs(s, g)) == _bits(py_f(*s, g))


def test_whitening_bits_match_pure_python_restatement(orc):
    """Step 2 / reading Q5: orc_init's base state = the key after N0 = 20000 steps of step 10, bit for bit."""
    for g, key in ((-1.0, KEY), (-0.06, (1.0, 2.0, 3.0, 4.0)), (-1.52, (-7.25, 0.001, 30.5, -12.0))):
        assert _bits(orc.ctx(key, g, 2, 4, 4).state) == _bits(py_rk4(key, g, N0))


def test_reconstruct_bits_match_pure_python_restatement(orc):
    rng = np.random.default_rng(11)
    for _ in range(3000):
        v = float(rng.uniform(-400, 400))
        hb = rng.integers(0, 256, 8, dtype=np.uint8).tobytes()
        assert _bits([orc.reconstruct(v, hb)]) == _bits([py_reconstruct(v, hb)])


def _six(d):
    return struct.pack("<d", d)[:6]


def replay_derive(S, gamma, n, w, h, H):
    """Steps 3-7 of SURVEY.md 8(c) replayed on the pure-Python restatement above (none of the oracle's
    primitives): reconstruction, LHCS_m records, skewed fetch, slicing, D-before-B order and layouts."""
    L = 2 * n
    s = tuple(py_reconstruct(float(S[v]), H[8 * v:8 * v + 8]) for v in range(4))
    IR = []
    for g in range(L):
        s = py_rk4(s, gamma, K_M)
        IR.append(s)
    ND = 3 * (h + w)
    D = np.zeros(ND, np.uint16)
    B = np.zeros(3 * w * h, np.uint8)
    for m in range(n):
        sys = []
        for q in range(2):
            g = 2 * m + q
            sys.append((IR[g][0], IR[(g + 1) % L][1], IR[(g + 2) % L][2], IR[(g + 3) % L][3]))
        d0, d1 = m * ND // n, (m + 1) * ND // n
        b0, b1 = (m * h // n) * w * 3, ((m + 1) * h // n) * w * 3

        def nxt():
            sys[0] = py_rk4_step(sys[0], gamma)
            sys[1] = py_rk4_step(sys[1], gamma)
            e0 = b"".join(_six(v) for v in sys[0])
            e1 = b"".join(_six(v) for v in sys[1])
            return bytes(a ^ b for a, b in zip(e0, e1))

        ds = b""
        for _ in range(-(-(d1 - d0) // 12)):
            ds += nxt()
        bs = b""
        for _ in range(-(-(b1 - b0) // 24)):
            bs += nxt()
        D[d0:d1] = np.frombuffer(ds, "<u2")[: d1 - d0]
        B[b0:b1] = np.frombuffer(bs, np.uint8)[: b1 - b0]
    return D, B.reshape(h, w, 3), np.array(IR)


@pytest.mark.parametrize("n,w,h", [(1, 4, 4), (2, 5, 7), (3, 8, 5), (4, 6, 3), (32, 16, 40)])
def test_derive_layout_replay(orc, n, w, h):
    ctx = orc.ctx(KEY, -1.0, n, w, h)
    S0 = ctx.state
    assert _bits(S0) == _bits(py_rk4(KEY, -1.0, N0))  # N0 whitening steps at init
    rng = np.random.default_rng(n)
    for frame in range(2):
        H = rng.integers(0, 256, 32, dtype=np.uint8).tobytes()
        S = ctx.state
        D, B, IR = ctx.derive(H, want_ir=True)
        D2, B2, IR2 = replay_derive(S, -1.0, n, w, h, H)
        assert IR.tobytes() == IR2.tobytes()
        assert (D == D2).all() and (B == B2).all()
        assert ctx.state.tobytes() == IR[-1].tobytes()  # x_2n..w_2n carried to the next frame


def _golden_derive_tiny():
    frames, cur = [], None
    for row in read_golden("derive_tiny.txt"):
        if row[0] == "H":
            cur = {"H": bytes.fromhex(row[1])}
            frames.append(cur)
        elif row[0] in ("S", "IR"):
            cur[row[0]] = struct.pack("<%dQ" % (len(row) - 1), *[int(x, 16) for x in row[1:]])
        elif row[0] == "D":
            cur["D"] = np.array([int(x, 16) for x in row[1:]], np.uint16)
        elif row[0] == "B":
            cur["B"] = np.frombuffer(bytes.fromhex(row[1]), np.uint8)
    return frames


def test_golden_derive_tiny_reproduced_by_oracle_and_by_restatement(orc):
    """tests/golden/derive_tiny.txt (n = 2, 5 x 7, two chained frames; written by tests/golden/make_derive_tiny.py
    from oracle/ alone): today's oracle still writes these bytes, and the pure-Python restatement -- started from
    the KEY, not from anything in the file -- arrives at the same base states, IR, D and B."""
    n, w, h, gamma = 2, 5, 7, -1.0
    frames = _golden_derive_tiny()
    assert len(frames) == 2 and frames[0]["D"].size == 3 * (h + w) and frames[0]["B"].size == 3 * w * h
    ctx = orc.ctx(KEY, gamma, n, w, h)
    S = py_rk4(KEY, gamma, N0)
    for fr in frames:
        assert ctx.state.tobytes() == fr["S"] == _bits(S)
        D, B, IR = ctx.derive(fr["H"], want_ir=True)
        assert IR.tobytes() == fr["IR"] and (D == fr["D"]).all() and (B.ravel() == fr["B"]).all()
        D2, B2, IR2 = replay_derive(S, gamma, n, w, h, fr["H"])
        assert IR2.tobytes() == fr["IR"] and (D2 == fr["D"]).all() and (B2.ravel() == fr["B"]).all()
        S = tuple(IR2[-1])


def test_worker_streams_are_not_shifted_copies(orc):
    """Reading Q4: with the skewed fetch and K_m = 16 the workers' byte streams are not
    time-shifted copies of one another (cross-worker byte equality at chance, 1/256)."""
    n, w, h = 8, 64, 64
    ctx = orc.ctx(KEY, -1.0, n, w, h)
    _, B = ctx.derive(bytes(range(32)))
    bands = B.reshape(n, -1)
    for lag in (0, 24, 48, 16 * 24, 32 * 24):
        eq = np.mean(bands[0][lag:] == bands[1][: bands.shape[1] - lag])
        assert eq < 0.02, (lag, eq)


def test_keystream_bytes_uniform(orc):
    """Every extracted byte position of the XORed stream is close to uniform (chi-square < 330
    ~ the 0.1 % point for 255 dof; PAPER.md:179 uses 293.25 = the 5 % point on real data)."""
    n, w, h = 4, 256, 192
    ctx = orc.ctx(KEY, -1.0, n, w, h)
    _, B = ctx.derive(bytes(32))
    b = B.ravel()
    for pos in range(6):
        sel = b[pos::6]
        cnt = np.bincount(sel, minlength=256)
        chi = ((cnt - sel.size / 256) ** 2 / (sel.size / 256)).sum()
        assert chi < 340, (pos, chi)


def test_O0_build_gives_identical_bits(orc):
    """P12 self-consistency: an -O0 build produces the same D, B and state bit patterns."""
    from oracle import oracle

    with tempfile.TemporaryDirectory() as td:
        lib0 = oracle.Lib(oracle.build("-O0", os.path.join(td, "liboracle_O0.so"), force=True))
        a, b = orc.ctx(KEY, -1.2, 5, 24, 17), lib0.ctx(KEY, -1.2, 5, 24, 17)
        for k in range(3):
            H = bytes((7 * k + i) & 255 for i in range(32))
            Da, Ba = a.derive(H)
            Db, Bb = b.derive(H)
            assert (Da == Db).all() and (Ba == Bb).all()
            assert a.state.tobytes() == b.state.tobytes()


def test_init_rejects_bad_gamma(orc):
    from oracle.oracle import OracleError

    for g in (-1.6, 0.0, float("nan")):
        with pytest.raises(OracleError):
            orc.ctx(KEY, g, 4, 8, 8)
