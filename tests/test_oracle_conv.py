"""Pins of the Eq. 1.1 oracle (oracle/wtide_oracle.py: trajectory_nodes, convolve_currents)
against what the paper and the mathematics fix.  CPU only.

Eq. 1.1: PAPER.md:35-39.  Each test names the plausible mistake it is meant to catch.
"""
import numpy as np
import pytest

from oracle import wtide_oracle as wo

SHAPE = (6, 5, 4)
LEN = (12.0, 7.5, 10.0)
NT = 16
DT = 0.01


def _rand_table(seed=1, shape=SHAPE, nt=NT):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape + (nt, 3))


def _one_carrier(pos, vel, q=1.0):
    pos = np.asarray(pos, np.float32).reshape(-1, 3)
    vel = np.asarray(vel, np.float32).reshape(-1, 3)
    return np.array([0, len(pos)], np.int64), pos, vel, np.array([q], np.float32)


def _conv(H, off, pos, vel, q, shape=SHAPE, lengths=LEN, nt=NT, v_w=1.0, toff=None):
    return wo.convolve_currents(H, shape, lengths, nt, DT, v_w, off, pos, vel, q, toff)


def test_single_step_on_a_node_reads_the_row_back():
    """A carrier sitting exactly on node (2,3,1) for one step: i[n] = -q H_row[n].v dt.
    Catches: wrong node/row indexing, wrong sign, missing dt or q, lag offset."""
    H = _rand_table()
    x = (2 * LEN[0] / SHAPE[0], 3 * LEN[1] / SHAPE[1], 1 * LEN[2] / SHAPE[2])
    v = np.array([3.0, -2.0, 0.5], np.float32)
    out = _conv(H, *_one_carrier([x], [v], q=-2.0))
    expect = -(-2.0) * (H[2, 3, 1] @ v.astype(np.float64)) * DT
    np.testing.assert_allclose(out[0], expect, rtol=1e-12, atol=1e-14)


def test_step_m_is_delayed_by_m_samples():
    """Second step only (first has zero velocity): output starts at n = 1 with lag 0.
    Catches: lag n-m reversed or off by one, causality (m <= n) wrong."""
    H = _rand_table(2)
    x = (2 * LEN[0] / SHAPE[0], 0.0, 0.0)
    v = np.array([1.0, 0.0, 0.0], np.float32)
    out = _conv(H, *_one_carrier([x, x], [0 * v, v]))
    assert out[0, 0] == 0.0
    np.testing.assert_allclose(out[0, 1:], -H[2, 0, 0, : NT - 1, 0] * DT, rtol=1e-12)


def test_position_independent_table_is_a_1d_causal_convolution():
    """north_star check 4: H(x,t) = h(t) c  =>  i = -(q/V_w) (h * (c.v)) dt, a textbook 1-D causal
    convolution (trilinear weights sum to 1).  np.convolve is the independent routine.
    Catches: weights not summing to one, dropped corner, wrong time quadrature."""
    rng = np.random.default_rng(3)
    h = rng.standard_normal(NT)
    c = np.array([0.3, -1.1, 0.7])
    H = np.broadcast_to(h[:, None] * c[None, :], SHAPE + (NT, 3)).copy()
    M = 9
    pos = rng.uniform(-20, 30, size=(M, 3))
    vel = rng.standard_normal((M, 3))
    off, p32, v32, q = _one_carrier(pos, vel, q=1.5)
    out = _conv(H, off, p32, v32, q, v_w=2.0)
    s = v32.astype(np.float64) @ c
    expect = -(1.5 / 2.0) * np.convolve(h, s)[:NT] * DT
    np.testing.assert_allclose(out[0], expect, rtol=1e-11, atol=1e-13)


def test_zero_resistance_table_gives_the_standard_ramo_current():
    """north_star check 1: H[0] = E(x)/dt, H[n>0] = 0  =>  i[n] = -q E(x[n]).v[n]/V_w.  E affine in x,
    sampled at the nodes, so that trilinear interpolation is exact inside the box.
    Catches: interpolation weights attached to the wrong corner, fraction of the wrong axis."""
    a = np.array([0.2, -0.4, 1.0])
    B = np.array([[0.05, 0.02, -0.01], [0.03, -0.07, 0.04], [-0.02, 0.01, 0.06]])
    xs = [np.arange(n) * l / n for n, l in zip(SHAPE, LEN)]
    X = np.stack(np.meshgrid(*xs, indexing="ij"), axis=-1)
    E = a + X @ B.T
    H = np.zeros(SHAPE + (NT, 3))
    H[..., 0, :] = E / DT
    rng = np.random.default_rng(4)
    M = NT
    hi = [l * (n - 1) / n for n, l in zip(SHAPE, LEN)]           # stay inside the un-wrapped cells
    pos = np.stack([rng.uniform(0, h_, M) for h_ in hi], axis=1).astype(np.float32)
    vel = rng.standard_normal((M, 3)).astype(np.float32)
    out = _conv(H, *_one_carrier(pos, vel, q=-1.0))
    e_at = a + pos.astype(np.float64) @ B.T
    expect = -(-1.0) * np.sum(e_at * vel.astype(np.float64), axis=1)
    np.testing.assert_allclose(out[0], expect, rtol=2e-6, atol=1e-7)   # fp32 index arithmetic (R24)


def test_linearity_and_time_shift():
    """Linear in q and v; k leading zero-velocity steps delay i by k samples.
    Catches: state carried between carriers, output not zero-initialised."""
    H = _rand_table(5)
    rng = np.random.default_rng(6)
    pos = rng.uniform(0, 10, size=(5, 3))
    vel = rng.standard_normal((5, 3))
    base = _conv(H, *_one_carrier(pos, vel, q=1.0))[0]
    np.testing.assert_allclose(_conv(H, *_one_carrier(pos, 2 * vel, q=-3.0))[0], -6 * base, rtol=1e-6, atol=1e-9)
    k = 3
    pos2 = np.concatenate([np.zeros((k, 3)), pos])
    vel2 = np.concatenate([np.zeros((k, 3)), vel])
    shifted = _conv(H, *_one_carrier(pos2, vel2))[0]
    assert np.all(shifted[:k] == 0)
    np.testing.assert_allclose(shifted[k:], base[: NT - k], rtol=1e-12, atol=1e-14)


def test_trajectory_nodes_wrap_clamp_and_exact_fraction():
    """R24 on hand-computed cases.  Catches: wrap of negative x, clamp of z, i1 at the top layer."""
    shape, lengths = (4, 4, 4), (8.0, 8.0, 8.0)       # inv = 0.5 exactly
    pos = np.array([[1.0, -1.0, 3.0],                 # u = (0.5, -0.5, 1.5)
                    [7.5, 8.5, 100.0],                # u = (3.75, 4.25, clamp 3)
                    [0.0, 0.0, -5.0]], np.float32)    # z clamps to 0
    i0, i1, f, fin = wo.trajectory_nodes(shape, lengths, pos)
    assert fin.all()
    assert i0.tolist() == [[0, 3, 1], [3, 0, 3], [0, 0, 0]]
    assert i1.tolist() == [[1, 0, 2], [0, 1, 3], [1, 1, 1]]
    np.testing.assert_array_equal(f, np.array([[0.5, 0.5, 0.5], [0.75, 0.25, 0.0], [0, 0, 0]], np.float32))
    _, _, _, fin = wo.trajectory_nodes(shape, lengths, np.array([[np.nan, 0, 0]], np.float32))
    assert not fin[0]


def _brute_force(H, shape, lengths, nt, dt, v_w, off, pos, vel, charge):
    """Eq. 1.1 as four nested pure-Python loops with its own index arithmetic (python floats on
    float32-rounded inputs)."""
    out = np.zeros((len(off) - 1, nt))
    for c in range(len(off) - 1):
        for n in range(nt):
            acc = 0.0
            for m in range(min(n + 1, off[c + 1] - off[c], nt)):
                s = off[c] + m
                idx, wts = [], []
                for a in range(3):
                    inv = float(np.float32(np.float64(shape[a]) / np.float64(lengths[a])))
                    u = float(np.float32(float(pos[s, a]) * inv))
                    if a == 2:
                        u = min(max(u, 0.0), shape[a] - 1.0)
                    i0 = int(np.floor(u))
                    fr = float(np.float32(u - i0))
                    if a < 2:
                        idx.append((i0 % shape[a], (i0 + 1) % shape[a]))
                    else:
                        idx.append((i0, min(i0 + 1, shape[a] - 1)))
                    wts.append((1.0 - fr, fr))
                for cx in (0, 1):
                    for cy in (0, 1):
                        for cz in (0, 1):
                            w = wts[0][cx] * wts[1][cy] * wts[2][cz]
                            for a in range(3):
                                acc += w * H[idx[0][cx], idx[1][cy], idx[2][cz], n - m, a] * float(vel[s, a])
            out[c, n] = -(float(charge[c]) / v_w) * acc * dt
    return out


def test_brute_force_direct_summation_tiny():
    """north_star check 3: literal quadruple loop on 6 carriers (ragged lengths incl. 0 and > nt),
    positions outside the box (wrap in x, y; clamp in z).  Catches any reorganisation error."""
    shape, lengths, nt = (4, 3, 3), (8.0, 4.5, 6.0), 6
    H = _rand_table(7, shape, nt)
    rng = np.random.default_rng(8)
    lens = [3, 0, 1, 9, 6, 2]
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    S = off[-1]
    pos = rng.uniform(-10, 20, size=(S, 3)).astype(np.float32)
    vel = rng.standard_normal((S, 3)).astype(np.float32)
    charge = rng.standard_normal(len(lens)).astype(np.float32)
    got = wo.convolve_currents(H, shape, lengths, nt, DT, 1.0, off, pos, vel, charge)
    ref = _brute_force(H, shape, lengths, nt, DT, 1.0, off, pos, vel, charge)
    np.testing.assert_allclose(got, ref, rtol=1e-10, atol=1e-13)
    toff = np.array([0, 2, 2, 6], np.int64)                    # a track with no carrier
    tr = wo.convolve_currents(H, shape, lengths, nt, DT, 1.0, off, pos, vel, charge, toff)
    np.testing.assert_allclose(tr[0], ref[0] + ref[1], rtol=1e-10, atol=1e-13)
    assert np.all(tr[1] == 0)
    np.testing.assert_allclose(tr[2], ref[2:].sum(0), rtol=1e-10, atol=1e-13)


def test_non_finite_step_is_skipped():
    H = _rand_table(9)
    pos = np.array([[1, 1, 1], [np.nan, 1, 1], [2, 2, 2]], np.float32)
    vel = np.ones((3, 3), np.float32)
    full = _conv(H, *_one_carrier(pos, vel))[0]
    pos_ok = pos.copy()
    pos_ok[1] = 0
    vel0 = vel.copy()
    vel0[1] = 0
    np.testing.assert_allclose(full, _conv(H, *_one_carrier(pos_ok, vel0))[0], rtol=1e-13)


def test_error_metric_definitions():
    ref = np.array([[0.0, 2.0, -4.0, 0.0]])
    tst = ref + np.array([[0.0, 0.0, 0.4, 0.0]])
    l2, mx = wo.current_error(tst, ref)
    assert l2 == pytest.approx(0.4 / (2.0 * 4.0))
    assert mx == pytest.approx(0.1)
