"""Pins for the float64 oracle (oracle/sdtw_oracle.c) against what the paper and the mathematics fix.

None of these re-uses the oracle's own recurrences: the references are brute-force enumeration of all
complete alignment paths (Def. 1-2, eq. 3-4), closed forms, exact integer
Delannoy counts, the gamma -> 0 sandwich around classic DTW (eq. 1), invariants of the expected alignment
E, central finite differences ("differentiable everywhere") and symmetries.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from paper_2404_12134_b200 import synth

HERE = os.path.dirname(os.path.abspath(__file__))


# ----------------------------------------------------------------------------- helpers (test-side, independent)
def all_paths(n, m):
    """Every complete alignment path from (0,0) to (n-1,m-1) with moves (0,1), (1,0), (1,1) (Def. 1)."""
    out = []

    def rec(i, j, acc):
        acc = acc + [(i, j)]
        if i == n - 1 and j == m - 1:
            out.append(acc)
            return
        if j + 1 < m:
            rec(i, j + 1, acc)
        if i + 1 < n:
            rec(i + 1, j, acc)
        if i + 1 < n and j + 1 < m:
            rec(i + 1, j + 1, acc)

    rec(0, 0, [])
    return out


def sqdist(x, z):
    x = np.asarray(x, np.float64).reshape(len(x), -1)
    z = np.asarray(z, np.float64).reshape(len(z), -1)
    return ((x[:, None, :] - z[None, :, :]) ** 2).sum(-1)


def brute_force(x, z, gamma):
    """value = -gamma log sum_A exp(-<A,D>/gamma) (eq. 3-4) and E = sum_A p(A) A, by enumeration."""
    D = sqdist(x, z)
    n, m = D.shape
    paths = all_paths(n, m)
    costs = np.array([sum(D[i, j] for i, j in p) for p in paths])
    cmin = costs.min()
    w = np.exp(-(costs - cmin) / gamma)
    value = cmin - gamma * math.log(w.sum())
    p = w / w.sum()
    E = np.zeros((n, m))
    for pk, path in zip(p, paths):
        for i, j in path:
            E[i, j] += pk
    return value, E, costs, paths


def delannoy(a, b):
    return sum(math.comb(a, k) * math.comb(b, k) * 2 ** k for k in range(min(a, b) + 1))


def dtw_minplus(D):
    """Classic DTW by the textbook min-plus DP in numpy (test-side re-statement of eq. 1)."""
    n, m = D.shape
    R = np.full((n + 1, m + 1), np.inf)
    R[0, 0] = 0.0
    for i in range(1, n + 1):
        for j in range(1, m + 1):
            R[i, j] = D[i - 1, j - 1] + min(R[i - 1, j - 1], R[i - 1, j], R[i, j - 1])
    return R[n, m]


def grad_from_E(E, x, z):
    x = np.asarray(x, np.float64).reshape(len(x), -1)
    z = np.asarray(z, np.float64).reshape(len(z), -1)
    return 2.0 * (E.sum(0)[:, None] * z - E.T @ x)


# ----------------------------------------------------------------------------- golden: path counts
def test_golden_delannoy_and_path_enumeration():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "delannoy.txt")) if l.strip() and l[0] != "#"]
    for a, b, v in rows:
        a, b, v = int(a), int(b), int(v)
        assert delannoy(a, b) == v
        if v <= 2000:
            assert len(all_paths(a + 1, b + 1)) == v


# ----------------------------------------------------------------------------- brute force (value, E, gradient)
@pytest.mark.parametrize("gamma", [1.0, 0.1, 0.01])
@pytest.mark.parametrize("shape", [(1, 1, 1), (1, 5, 1), (4, 1, 2), (2, 2, 1), (3, 4, 1), (5, 6, 1), (6, 5, 2), (6, 6, 3)])
def test_brute_force_value_E_grad(oracle, gamma, shape):
    n, m, d = shape
    rng = np.random.default_rng(1000 * n + 10 * m + d)
    x = rng.normal(size=(n, d))
    z = rng.normal(size=(m, d))
    v_bf, E_bf, _, _ = brute_force(x, z, gamma)
    r = oracle.pair(x, z, gamma, want_grad=True, want_E=True, want_R=True)
    assert abs(r["value"] - v_bf) <= 1e-12 * max(1.0, abs(v_bf))
    assert np.abs(r["E"] - E_bf).max() <= 1e-12
    assert np.abs(r["grad"] - grad_from_E(E_bf, x, z)).max() <= 1e-11
    # the probability-flow form of the reverse DP must give the same E
    D = oracle.cost_matrix(x, z)
    assert np.abs(D - sqdist(x, z)).max() <= 1e-14
    En = oracle.backward_E_normalised(D, r["R"], gamma)
    assert np.abs(En - E_bf).max() <= 1e-12
    # checkpointed mode, same numbers bitwise
    rc = oracle.pair(x, z, gamma, mode="checkpointed")
    assert rc["value"] == r["value"] and np.array_equal(rc["grad"], r["grad"])


def test_R_border_and_every_cell_against_brute_force(oracle):
    """r_00 = 0, r_i0 = r_0j = inf (eq. 5) and every interior r_ij = soft-min over paths to (i,j)."""
    rng = np.random.default_rng(7)
    x, z, gamma = rng.normal(size=4), rng.normal(size=5), 0.3
    R = oracle.pair(x, z, gamma, want_R=True)["R"]
    assert R[0, 0] == 0.0 and np.all(np.isinf(R[0, 1:6])) and np.all(np.isinf(R[1:5, 0]))
    for i in range(1, 5):
        for j in range(1, 6):
            v, _, _, _ = brute_force(x[:i], z[:j], gamma)
            assert abs(R[i, j] - v) < 1e-12


# ----------------------------------------------------------------------------- closed forms
def test_single_cell_and_single_row_column(oracle):
    rng = np.random.default_rng(3)
    for d in (1, 3):
        x = rng.normal(size=(1, d))
        z = rng.normal(size=(1, d))
        r = oracle.pair(x, z, 0.5, want_E=True)
        assert abs(r["value"] - ((x - z) ** 2).sum()) < 1e-15
        assert r["E"].tolist() == [[1.0]]
        assert np.allclose(r["grad"], 2 * (z - x), atol=1e-15)
        # n = 1: a single path through every column
        z = rng.normal(size=(7, d))
        r = oracle.pair(x, z, 0.5, want_E=True)
        assert abs(r["value"] - sqdist(x, z).sum()) < 1e-13
        assert np.abs(r["E"] - 1.0).max() < 1e-13 and r["E"].shape == (1, 7)
        assert np.allclose(r["grad"], 2 * (z - x), atol=1e-14)
        # m = 1
        xx = rng.normal(size=(6, d))
        zz = rng.normal(size=(1, d))
        r = oracle.pair(xx, zz, 0.5, want_E=True)
        assert abs(r["value"] - sqdist(xx, zz).sum()) < 1e-13
        assert np.abs(r["E"] - 1.0).max() < 1e-13 and r["E"].shape == (6, 1)
        assert np.allclose(r["grad"], 2 * (6 * zz - xx.sum(0, keepdims=True)), atol=1e-13)


@pytest.mark.parametrize("n,m", [(1, 1), (3, 3), (6, 9), (40, 55)])
def test_zero_cost_closed_form_delannoy(oracle, n, m):
    """x == z == const => D == 0: value = -gamma ln Del(n-1,m-1), E_ij = Del(i-1,j-1) Del(n-i,m-j)/Del(n-1,m-1)."""
    gamma = 0.7
    x = np.full(n, 0.25)
    z = np.full(m, 0.25)
    r = oracle.pair(x, z, gamma, want_E=True)
    tot = delannoy(n - 1, m - 1)
    assert abs(r["value"] + gamma * math.log(tot)) <= 1e-9 * max(1.0, gamma * math.log(tot))
    Eex = np.array([[float(Fraction(delannoy(i, j) * delannoy(n - 1 - i, m - 1 - j), tot)) for j in range(m)]
                    for i in range(n)])
    assert np.abs(r["E"] - Eex).max() <= 1e-9
    assert np.abs(r["grad"]).max() == 0.0


@pytest.mark.parametrize("n,m", [(4, 4), (7, 5), (12, 20)])
def test_constant_cost_closed_form(oracle, n, m):
    """x == a, z == b: every cell costs delta; paths with k diagonal moves have n+m-1-k cells and there are
    (n+m-2-k)! / (k! (n-1-k)! (m-1-k)!) of them."""
    a, b, gamma = 0.3, -0.4, 0.25
    delta = (a - b) ** 2
    terms = []
    mean_len_num = 0.0
    for k in range(min(n, m)):
        cnt = math.factorial(n + m - 2 - k) // (math.factorial(k) * math.factorial(n - 1 - k) * math.factorial(m - 1 - k))
        terms.append((cnt, n + m - 1 - k))
    Zsum = sum(c * math.exp(-delta * L / gamma) for c, L in terms)
    v_ex = -gamma * math.log(Zsum)
    mean_len = sum(c * math.exp(-delta * L / gamma) * L for c, L in terms) / Zsum
    r = oracle.pair(np.full(n, a), np.full(m, b), gamma, want_E=True)
    assert abs(r["value"] - v_ex) <= 1e-9 * abs(v_ex)
    assert abs(r["E"].sum() - mean_len) <= 1e-9 * mean_len
    assert abs(r["grad"].sum() - 2 * (b - a) * mean_len) <= 1e-9 * abs(2 * (b - a) * mean_len)


# ----------------------------------------------------------------------------- gamma -> 0 (eq. 3 first case, eq. 1)
def test_gamma_to_zero_sandwich_and_monotone(oracle):
    rng = np.random.default_rng(11)
    for n, m, d in [(5, 6, 1), (30, 41, 1), (25, 20, 2)]:
        x = rng.normal(size=(n, d))
        z = rng.normal(size=(m, d))
        D = sqdist(x, z)
        dtw = dtw_minplus(D)
        assert abs(oracle.dtw(x, z) - dtw) <= 1e-12 * max(1, dtw)
        if n * m <= 36:
            _, _, costs, _ = brute_force(x, z, 1.0)
            assert abs(costs.min() - dtw) < 1e-12          # eq. 1 by enumeration
        prev = None
        for gamma in [1.0, 0.3, 0.1, 0.01, 1e-3, 1e-5]:
            v = oracle.pair(x, z, gamma, want_grad=False)["value"]
            lo = dtw - gamma * math.log(delannoy(n - 1, m - 1))
            assert lo - 1e-9 <= v <= dtw + 1e-12
            if prev is not None:
                assert v >= prev - 1e-12                   # d value / d gamma = -entropy <= 0
            prev = v
        assert abs(prev - dtw) <= 1e-5 * math.log(delannoy(n - 1, m - 1)) + 1e-12


# ----------------------------------------------------------------------------- invariants of E, free-energy identity
@pytest.mark.parametrize("gamma", [1.0, 0.1, 0.01])
def test_E_invariants_and_free_energy_identity(oracle, gamma):
    rng = np.random.default_rng(5)
    n, m = 60, 70
    t = np.linspace(0, 1, n)
    x = np.sin(6 * t) + 0.05 * rng.normal(size=n)
    z = np.sin(6 * np.linspace(0, 1, m) ** 1.2)
    r = oracle.pair(x, z, gamma, want_E=True, want_R=True)
    E, R = r["E"], r["R"]
    assert E.min() >= -1e-15 and E.max() <= 1 + 1e-12
    assert abs(E[0, 0] - 1) < 1e-12 and abs(E[-1, -1] - 1) < 1e-12
    assert E.sum(1).min() >= 1 - 1e-12 and E.sum(0).min() >= 1 - 1e-12
    assert max(n, m) - 1e-9 <= E.sum() <= n + m - 1 + 1e-9
    # value = sum_s E[s] (D[s] - gamma H_s), H_s = entropy of softmax(-R[pred(s)]/gamma)   (test-side formula)
    D = sqdist(x, z)
    tot = 0.0
    for i in range(1, n + 1):
        for j in range(1, m + 1):
            pr = np.array([R[i - 1, j - 1], R[i - 1, j], R[i, j - 1]])
            pr = pr[np.isfinite(pr)]
            w = np.exp(-(pr - pr.min()) / gamma)
            w /= w.sum()
            H = -(w[w > 0] * np.log(w[w > 0])).sum()
            tot += E[i - 1, j - 1] * (D[i - 1, j - 1] - gamma * H)
    assert abs(tot - r["value"]) <= 1e-9 * max(1.0, abs(r["value"]))
    # the two reverse-DP forms agree
    En = oracle.backward_E_normalised(D, R, gamma)
    assert np.abs(En - E).max() < 1e-10


# ----------------------------------------------------------------------------- finite differences
@pytest.mark.parametrize("gamma,d", [(1.0, 1), (0.1, 1), (0.1, 3), (0.01, 1)])
def test_gradient_finite_differences(oracle, gamma, d):
    rng = np.random.default_rng(21 + d)
    N, m = 3, 17
    lens = [15, 19, 12]
    xs = [np.cumsum(rng.normal(size=(n, d)), 0) * 0.2 for n in lens]
    X = np.concatenate(xs).astype(np.float32)
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    Z = (np.cumsum(rng.normal(size=(m, d)), 0) * 0.2).astype(np.float32)
    vals, G = oracle.value_grad(Z, X, off, gamma)

    def obj(Zd):
        return sum(oracle.pair(xk.astype(np.float32).astype(np.float64), Zd, gamma, want_grad=False)["value"] for xk in xs)

    Zd = Z.astype(np.float64)
    assert abs(obj(Zd) - vals.sum()) < 1e-10 * max(1, abs(vals.sum()))
    for j in range(m):
        for c in range(d):
            h = 1e-5 * max(1.0, abs(Zd[j, c]))
            Zp, Zm = Zd.copy(), Zd.copy()
            Zp[j, c] += h
            Zm[j, c] -= h
            fd = (obj(Zp) - obj(Zm)) / (2 * h)
            assert abs(fd - G[j, c]) <= 1e-6 * max(1.0, abs(G[j, c])), (j, c, fd, G[j, c])


# ----------------------------------------------------------------------------- symmetries, scaling, additivity
def test_symmetries_scaling_additivity(oracle):
    rng = np.random.default_rng(9)
    n, m, d, gamma = 14, 11, 2, 0.2
    x = rng.normal(size=(n, d))
    z = rng.normal(size=(m, d))
    a = oracle.pair(x, z, gamma, want_E=True)
    b = oracle.pair(z, x, gamma, want_E=True)
    assert abs(a["value"] - b["value"]) < 1e-12 and np.abs(a["E"] - b["E"].T).max() < 1e-12
    c = oracle.pair(x[::-1], z[::-1], gamma, want_E=True)
    assert abs(a["value"] - c["value"]) < 1e-12 and np.abs(a["E"] - c["E"][::-1, ::-1]).max() < 1e-12
    s = oracle.pair(x + 3.0, z + 3.0, gamma, want_E=True)
    assert abs(a["value"] - s["value"]) < 1e-11
    sc = 1.7
    e = oracle.pair(sc * x, sc * z, gamma * sc * sc, want_E=True)
    assert abs(e["value"] - sc * sc * a["value"]) < 1e-11 and np.abs(e["E"] - a["E"]).max() < 1e-11
    # additivity over pairs: summed call == sum of single-pair calls
    lens = [9, 14, 6, 11]
    X = rng.normal(size=(sum(lens), d)).astype(np.float32)
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    Z = z.astype(np.float32)
    vals, G = oracle.value_grad(Z, X, off, gamma)
    Gs = np.zeros_like(G)
    for k in range(4):
        r = oracle.pair(X[off[k]:off[k + 1]].astype(np.float64), Z.astype(np.float64), gamma)
        assert abs(vals[k] - r["value"]) < 1e-13 * max(1, abs(r["value"]))
        Gs += r["grad"]
    assert np.abs(G - Gs).max() < 1e-12
    # thread count must not change anything (fixed k order of the final sum)
    vals1, G1 = oracle.value_grad(Z, X, off, gamma, nthreads=1)
    assert np.array_equal(vals, vals1) and np.array_equal(G, G1)


# ----------------------------------------------------------------------------- checkpointed mode == full mode, cfg 2
def test_checkpointed_mode_bitwise_on_medium_config(oracle):
    data = synth.make(2)
    off = data["offsets"][:5]            # 4 pairs of ~1000 x 1000 are enough to cover block edges
    X = data["X"][:off[-1]]
    v0, g0 = oracle.value_grad(data["Z0"], X, off, data["cfg"].gamma, mode="full")
    v1, g1 = oracle.value_grad(data["Z0"], X, off, data["cfg"].gamma, mode="checkpointed")
    assert np.array_equal(v0, v1) and np.array_equal(g0, g1)
    assert np.all(np.isfinite(g0)) and np.abs(g0).max() > 0


# ----------------------------------------------------------------------------- barycenter loop
def test_barycenter_tiny_config_descends_and_matches_manual_loop(oracle):
    data = synth.make(1)
    cfg = data["cfg"]
    Z, vals, obj = oracle.barycenter(data["Z0"], data["X"], data["offsets"], cfg.gamma, cfg.iters, cfg.step)
    assert len(obj) == cfg.iters and np.all(np.diff(obj) < 0)          # monotone descent at step 0.01 (cfg 1)
    # first objective / first update reproduce a value_grad call at Z0
    v0, g0 = oracle.value_grad(data["Z0"], data["X"], data["offsets"], cfg.gamma)
    assert abs(obj[0] - v0.sum()) < 1e-12 * abs(v0.sum())
    Z1, _, _ = oracle.barycenter(data["Z0"], data["X"], data["offsets"], cfg.gamma, 1, cfg.step)
    assert np.abs(Z1 - (data["Z0"].astype(np.float64) - cfg.step * g0)).max() < 1e-15
    # iters = 0 leaves Z0 untouched
    Zn, _, _ = oracle.barycenter(data["Z0"], data["X"], data["offsets"], cfg.gamma, 0, cfg.step)
    assert np.array_equal(Zn, data["Z0"].astype(np.float64))
    # the GD fixed point lowers the objective relative to the Euclidean-mean start
    vend, _ = oracle.value_grad(Z.astype(np.float32), data["X"], data["offsets"], cfg.gamma, want_grad=False)
    assert vend.sum() < obj[0]


# ----------------------------------------------------------------------------- Sakoe-Chiba band (Table 1)
def brute_force_banded(x, z, gamma, band):
    """Soft-min over the complete alignment paths that stay inside |i - j| <= band (reading C18), by enumeration."""
    D = sqdist(x, z)
    n, m = D.shape
    paths = [p for p in all_paths(n, m) if all(abs(i - j) <= band for i, j in p)]
    costs = np.array([sum(D[i, j] for i, j in p) for p in paths])
    cmin = costs.min()
    w = np.exp(-(costs - cmin) / gamma)
    value = cmin - gamma * math.log(w.sum())
    E = np.zeros((n, m))
    for pk, path in zip(w / w.sum(), paths):
        for i, j in path:
            E[i, j] += pk
    return value, E, len(paths)


@pytest.mark.parametrize("gamma", [1.0, 0.05])
@pytest.mark.parametrize("shape_band", [((5, 5, 1), 0), ((5, 5, 2), 1), ((6, 6, 1), 2), ((6, 4, 1), 2), ((4, 6, 2), 2),
                                        ((4, 6, 1), 3), ((6, 5, 1), 1), ((6, 6, 1), 5), ((1, 3, 1), 2), ((3, 1, 1), 2)])
def test_band_brute_force_value_E_grad(oracle, gamma, shape_band):
    (n, m, d), band = shape_band
    rng = np.random.default_rng(77 * n + 7 * m + d + band)
    x = rng.normal(size=(n, d))
    z = rng.normal(size=(m, d))
    v_bf, E_bf, npaths = brute_force_banded(x, z, gamma, band)
    assert npaths >= 1
    r = oracle.pair(x, z, gamma, want_E=True, want_R=True, band=band)
    assert abs(r["value"] - v_bf) <= 1e-12 * max(1.0, abs(v_bf))
    assert np.abs(r["E"] - E_bf).max() <= 1e-12
    assert np.abs(r["grad"] - grad_from_E(E_bf, x, z)).max() <= 1e-11
    # cells outside the band: r = +inf, E = 0 exactly
    ii, jj = np.indices((n, m))
    out = np.abs(ii - jj) > band
    assert np.all(np.isinf(r["R"][1:n + 1, 1:m + 1][out])) and np.all(r["E"][out] == 0.0)
    # checkpointed mode: same bits
    rc = oracle.pair(x, z, gamma, mode="checkpointed", band=band)
    assert rc["value"] == r["value"] and np.array_equal(rc["grad"], r["grad"])


def test_band_limits_and_infeasible(oracle):
    rng = np.random.default_rng(5)
    n, m, d, gamma = 17, 13, 2, 0.3
    x = rng.normal(size=(n, d))
    z = rng.normal(size=(m, d))
    free = oracle.pair(x, z, gamma, want_E=True)
    wide = oracle.pair(x, z, gamma, want_E=True, band=max(n, m) - 1)       # every cell admissible
    assert wide["value"] == free["value"] and np.array_equal(wide["E"], free["E"])
    # a narrower band removes paths: the soft-min over fewer paths is larger (eq. 3-4), and monotone in the band
    vals = [oracle.pair(x, z, gamma, want_grad=False, band=b)["value"] for b in range(n - m, n)]
    assert all(a >= b - 1e-12 for a, b in zip(vals, vals[1:])) and vals[0] > free["value"]
    # band 0 with n == m leaves the single diagonal path: value = trace(D), E = I, g_j = 2 (z_j - x_j)
    xs = rng.normal(size=(9, d))
    zs = rng.normal(size=(9, d))
    r0 = oracle.pair(xs, zs, gamma, want_E=True, band=0)
    assert abs(r0["value"] - np.trace(sqdist(xs, zs))) < 1e-12
    assert np.abs(r0["E"] - np.eye(9)).max() < 1e-12 and np.abs(r0["grad"] - 2 * (zs - xs)).max() < 1e-11
    # |n - m| > band: no complete path inside the band -> rejected
    with pytest.raises(RuntimeError):
        oracle.pair(x, z, gamma, band=n - m - 1)
    # finite differences of the banded value
    band = 6
    g = oracle.pair(x, z, gamma, band=band)["grad"]
    for (j, c) in [(0, 0), (5, 1), (12, 0)]:
        h = 1e-6
        zp, zm = z.copy(), z.copy()
        zp[j, c] += h
        zm[j, c] -= h
        fd = (oracle.pair(x, zp, gamma, want_grad=False, band=band)["value"] -
              oracle.pair(x, zm, gamma, want_grad=False, band=band)["value"]) / (2 * h)
        assert abs(fd - g[j, c]) <= 1e-6 * max(1.0, abs(g[j, c]))


# ----------------------------------------------------------------------------- eq. 7 weights lambda_k / n_k
def test_weighted_objective_and_gradient(oracle):
    rng = np.random.default_rng(21)
    d, m, gamma = 2, 12, 0.4
    lens = [9, 15, 12, 7]
    X = rng.normal(size=(sum(lens), d)).astype(np.float32)
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    Z = rng.normal(size=(m, d)).astype(np.float32)
    lam = np.array([1.0, 0.5, 2.0, 1.5])
    w = lam / np.array(lens)                                    # eq. 7: lambda_i / m_i
    vals, G, obj = oracle.value_grad(Z, X, off, gamma, weights=w, want_objective=True)
    vals1, _ = oracle.value_grad(Z, X, off, gamma)
    assert np.array_equal(vals, vals1)                          # per-pair values stay unweighted
    Gs = np.zeros_like(G)
    for k in range(4):
        r = oracle.pair(X[off[k]:off[k + 1]].astype(np.float64), Z.astype(np.float64), gamma)
        Gs += w[k] * r["grad"]
    assert np.abs(G - Gs).max() < 1e-13 and abs(obj - float(w @ vals)) < 1e-13
    # all-ones weights == the unweighted call, bitwise
    v2, G2 = oracle.value_grad(Z, X, off, gamma, weights=np.ones(4))
    _, G3 = oracle.value_grad(Z, X, off, gamma)
    assert np.array_equal(G2, G3)
    # finite differences of the weighted objective
    for (j, c) in [(0, 1), (6, 0), (11, 1)]:
        h = 1e-3                                                # Z is fp32 at this interface: exact fp32 steps
        Zp, Zm = Z.copy(), Z.copy()
        Zp[j, c] += np.float32(h)
        Zm[j, c] -= np.float32(h)
        op = oracle.value_grad(Zp, X, off, gamma, want_grad=False, weights=w, want_objective=True)[2]
        om = oracle.value_grad(Zm, X, off, gamma, want_grad=False, weights=w, want_objective=True)[2]
        fd = (op - om) / (float(Zp[j, c]) - float(Zm[j, c]))
        assert abs(fd - G[j, c]) <= 2e-5 * max(1.0, abs(G[j, c]))
    # descent on the weighted, banded objective: first update = Z0 - step * weighted gradient
    Z1, _, o1 = oracle.barycenter(Z, X, off, gamma, 1, 0.05, weights=w, band=8)
    vb, Gb, ob = oracle.value_grad(Z, X, off, gamma, weights=w, band=8, want_objective=True)
    assert np.abs(Z1 - (Z.astype(np.float64) - 0.05 * Gb)).max() < 1e-15 and abs(o1[0] - ob) < 1e-13


# ----------------------------------------------------------------------------- Def. 8 / eq. 8: d_score = DTW / |pi|
def brute_force_dtw(x, z):
    """eq. 1 by enumeration: (min cost, the cost-sorted list of (cost, path))."""
    D = sqdist(x, z)
    paths = all_paths(*D.shape)
    costs = np.array([sum(D[i, j] for i, j in p) for p in paths])
    order = np.argsort(costs)
    return costs[order[0]], [(costs[k], paths[k]) for k in order]


@pytest.mark.parametrize("shape", [(1, 1, 1), (1, 4, 2), (5, 1, 1), (3, 3, 1), (4, 6, 1), (6, 5, 2), (6, 6, 3)])
def test_dtw_path_length_brute_force(oracle, shape):
    n, m, d = shape
    rng = np.random.default_rng(31 * n + 5 * m + d)
    x = rng.normal(size=(n, d))
    z = rng.normal(size=(m, d))
    best, ranked = brute_force_dtw(x, z)
    assert len(ranked) == 1 or ranked[1][0] - ranked[0][0] > 1e-9          # the optimal path is unique on this draw
    v, ln, path = oracle.dtw_path(x, z, want_path=True)
    assert abs(v - best) <= 1e-12 * max(1.0, best) and ln == len(ranked[0][1])
    assert [(i - 1, j - 1) for i, j in path.tolist()] == ranked[0][1]      # and it is THE path, cell by cell
    assert max(n, m) <= ln <= n + m - 1
    assert abs(v - oracle.dtw(x, z)) == 0.0 and abs(v - dtw_minplus(sqdist(x, z))) <= 1e-12
    # float32-decision mirror: same path length, value within float32 round-off
    v32, l32, s32 = oracle.dtw_score(z.astype(np.float32), x.astype(np.float32), np.array([0, n]))
    v64, l64 = oracle.dtw_path(x.astype(np.float32).astype(np.float64), z.astype(np.float32).astype(np.float64))
    assert l32[0] == l64 and abs(v32[0] - v64) <= 1e-5 * max(1.0, v64)
    assert s32[0] == np.float32(v32[0]) / np.float32(l32[0])


def test_dtw_score_ties_special_cases_and_batch(oracle):
    # all costs equal (constant series): every path is optimal; the stated tie-break (diagonal, then up, then left)
    # walks the diagonal and then one edge: |pi| = max(n, m), DTW = (a - b)^2 |pi|
    for n, m in [(5, 5), (4, 9), (9, 4), (1, 6), (7, 1)]:
        x = np.full((n, 1), 0.5, np.float32)
        z = np.full((m, 1), 0.25, np.float32)
        v, ln, sc = oracle.dtw_score(z, x, np.array([0, n]))
        assert ln[0] == max(n, m) and v[0] == np.float32(0.0625 * max(n, m)) and sc[0] == np.float32(0.0625)
        v64, l64, path = oracle.dtw_path(x, z, want_path=True)
        assert l64 == max(n, m) and abs(v64 - 0.0625 * max(n, m)) < 1e-15
        steps = np.diff(path, axis=0)
        assert np.all((steps >= 0) & (steps <= 1)) and np.all(steps.sum(1) >= 1)       # a valid alignment path (Def. 1)
        assert tuple(path[0]) == (1, 1) and tuple(path[-1]) == (n, m)
    # identical series: DTW = 0 along the diagonal, |pi| = n
    rng = np.random.default_rng(3)
    x = rng.normal(size=(40, 2)).astype(np.float32)
    v, ln, sc = oracle.dtw_score(x, x, np.array([0, 40]))
    assert v[0] == 0.0 and ln[0] == 40 and sc[0] == 0.0
    # a series and its copy with every sample repeated twice: DTW = 0, |pi| = 2n (each z_j matched to two rows)
    v, ln, sc = oracle.dtw_score(x, np.repeat(x, 2, axis=0), np.array([0, 80]))
    assert v[0] == 0.0 and ln[0] == 80
    # batch == single calls; soft-DTW sandwich (eq. 3: gamma -> 0) ties the hard value to the pinned soft one
    data = synth.make(1)
    cfg = data["cfg"]
    v, ln, sc = oracle.dtw_score(data["Z0"], data["X"], data["offsets"])
    for k in range(cfg.N):
        a, b = data["offsets"][k], data["offsets"][k + 1]
        vk, lk, sk = oracle.dtw_score(data["Z0"], data["X"][a:b], np.array([0, b - a]))
        assert vk[0] == v[k] and lk[0] == ln[k] and sk[0] == sc[k]
        v64, l64 = oracle.dtw_path(data["X"][a:b].astype(np.float64), data["Z0"].astype(np.float64))
        assert abs(v[k] - v64) <= 1e-5 * v64 and ln[k] == l64
        soft = oracle.pair(data["X"][a:b].astype(np.float64), data["Z0"].astype(np.float64), 1e-3, want_grad=False)["value"]
        assert v64 - 1e-3 * math.log(delannoy(b - a - 1, cfg.m - 1)) - 1e-9 <= soft <= v64 + 1e-9


# ----------------------------------------------------------------------------- eq. 2: Sub-DTW (Step 1's primitive)
@pytest.mark.parametrize("shape", [(1, 1, 1), (6, 1, 1), (1, 4, 1), (7, 3, 1), (9, 4, 2), (12, 5, 1), (5, 7, 2)])
def test_subdtw_is_min_over_subsequences(oracle, shape):
    """eq. 2, second form: Sub-DTW(X, Y) = min_{a <= b} DTW(X, Y[a:b]) -- brute force over every (a, b) with the
    (separately pinned) classic DTW, and over every subsequence alignment path (first form) on the small cases."""
    n, m, d = shape                       # n = window length (free ends), m = reference length (fully traversed)
    rng = np.random.default_rng(17 * n + m + d)
    y = rng.normal(size=(n, d))
    z = rng.normal(size=(m, d))
    table = {(a, b): dtw_minplus(sqdist(y[a:b + 1], z)) for a in range(n) for b in range(a, n)}
    best = min(table.values())
    v, a, b = oracle.subdtw(y, z)
    assert abs(v - best) <= 1e-12 * max(1.0, best)
    assert 0 <= a <= b < n and abs(table[(a, b)] - best) <= 1e-12 * max(1.0, best)     # (a*, b*) attains the minimum
    assert sorted(table.values())[1] - best > 1e-9 if len(table) > 1 else True        # and it is unique on this draw
    if n * m <= 36:                       # first form: all paths with i_1 = 1, i_k = M along the reference
        D = sqdist(y, z)
        costs = []
        for a0 in range(n):
            for b0 in range(a0, n):
                for path in all_paths(b0 - a0 + 1, m):
                    costs.append(sum(D[a0 + i, j] for i, j in path))
        assert abs(min(costs) - v) <= 1e-12 * max(1.0, v)
    # float32-decision mirror: same (a*, b*), value within float32 round-off
    v32, a32, b32 = oracle.subdtw_f32(z.astype(np.float32), y.astype(np.float32), np.array([0, n]))
    v64, a64, b64 = oracle.subdtw(y.astype(np.float32).astype(np.float64), z.astype(np.float32).astype(np.float64))
    assert (a32[0], b32[0]) == (a64, b64) and abs(v32[0] - v64) <= 1e-5 * max(1.0, v64)


def test_subdtw_embedded_copy_ties_and_batch(oracle):
    rng = np.random.default_rng(8)
    z = rng.normal(size=(30, 2)).astype(np.float32)
    y = np.concatenate([3 + rng.normal(size=(17, 2)), z, 3 + rng.normal(size=(25, 2))]).astype(np.float32)
    v, a, b = oracle.subdtw_f32(z, y, np.array([0, len(y)]))
    assert v[0] == 0.0 and (a[0], b[0]) == (17, 46)                    # the embedded copy is found exactly
    v64, a64, b64 = oracle.subdtw(y, z)
    assert v64 == 0.0 and (a64, b64) == (17, 46)
    # a time-stretched copy (every sample twice): still cost 0, spanning the 2 m stretched samples
    y2 = np.concatenate([5 + rng.normal(size=(9, 2)), np.repeat(z, 2, axis=0), 5 + rng.normal(size=(4, 2))]).astype(np.float32)
    v, a, b = oracle.subdtw_f32(z, y2, np.array([0, len(y2)]))
    assert v[0] == 0.0 and 9 <= a[0] <= 10 and 67 <= b[0] <= 68        # either repeated end sample may be dropped (ties)
    assert oracle.subdtw(y2, z) == (0.0, a[0], b[0])
    # all cells tie (constant series): every path of m cells costs the same; the smallest b* is row 0 (the whole
    # reference matched to the first sample), so a* = b* = 0
    yc = np.full((12, 1), 0.5, np.float32)
    zc = np.full((5, 1), 0.25, np.float32)
    v, a, b = oracle.subdtw_f32(zc, yc, np.array([0, 12]))
    v64, a64, b64 = oracle.subdtw(yc, zc)
    assert (a[0], b[0]) == (a64, b64) == (0, 0) and v[0] == np.float32(5 * 0.0625)
    # Sub-DTW <= DTW of the whole window (the whole window is one of the subsequences), and batch == single calls
    data = synth.make(1)
    v, a, b = oracle.subdtw_f32(data["Z0"], data["X"], data["offsets"])
    dv, _, _ = oracle.dtw_score(data["Z0"], data["X"], data["offsets"])
    assert np.all(v <= dv)
    for k in range(data["cfg"].N):
        lo, hi = data["offsets"][k], data["offsets"][k + 1]
        vk, ak, bk = oracle.subdtw_f32(data["Z0"], data["X"][lo:hi], np.array([0, hi - lo]))
        assert (vk[0], ak[0], bk[0]) == (v[k], a[k], b[k])


# ----------------------------------------------------------------------------- backtracking descent (NEXT-3, reading C22)
def test_backtracking_descent_armijo_conditions(oracle):
    data = synth.make(1)
    cfg = data["cfg"]
    Z0, X, off = data["Z0"], data["X"], data["offsets"]
    step0, shrink, c1, iters = 0.64, 0.5, 1e-4, 5
    Z, vals, obj, steps, trials = oracle.barycenter_backtracking(Z0, X, off, cfg.gamma, iters, step0, shrink, c1)
    assert np.all(np.diff(obj) < 0) and len(obj) == iters + 1 and np.all(trials >= 1)
    # replay the first iteration with independent value_grad calls: every rejected step violates the Armijo
    # condition, the accepted one satisfies it, and Z moved by exactly that step (float32 Z0 is exact in float64)
    v0, G0 = oracle.value_grad(Z0, X, off, cfg.gamma)
    f0, gg = v0.sum(), float((G0 ** 2).sum())
    assert abs(obj[0] - f0) < 1e-12 * abs(f0)
    t = step0
    for tr in range(trials[0]):
        Zt = Z0.astype(np.float64) - t * G0
        Z1, _, o1 = oracle.barycenter(Z0, X, off, cfg.gamma, 2, t)      # o1[1] = f(Z0 - t G0), evaluated in float64
        ok = o1[1] <= f0 - c1 * t * gg
        assert ok == (tr == trials[0] - 1), (tr, t, o1[1], f0)
        if ok:
            assert t == steps[0] and abs(o1[1] - obj[1]) < 1e-12 * abs(f0)
        t *= shrink
    # a step that is always accepted reproduces the fixed-step loop bit for bit; a hopeless one stops the descent
    Zf, _, of = oracle.barycenter(Z0, X, off, cfg.gamma, 3, 0.01)
    Zb, _, ob, sb, tb = oracle.barycenter_backtracking(Z0, X, off, cfg.gamma, 3, 0.01, shrink, 0.0)
    assert np.array_equal(Zf, Zb) and np.array_equal(of, ob[:3]) and np.all(sb == 0.01) and np.all(tb == 1)
    Zs, _, os_, ss, ts = oracle.barycenter_backtracking(Z0, X, off, cfg.gamma, 3, 50.0, shrink, c1, max_trials=1)
    assert np.array_equal(Zs, Z0.astype(np.float64)) and np.all(ss == 0) and ts[0] == 1 and np.all(os_ == os_[0])


def test_descent_driven_one_evaluation_at_a_time_is_the_c_loop_bitwise(oracle):
    """oracle.value_grad_f64z (the evaluation at a float64 barycenter) driven by Z <- Z - step G in numpy reproduces
    oracle.barycenter bit for bit: that is how tests/golden/make_fullsize_refs.py writes the full-size references."""
    from paper_2404_12134_b200 import synth
    for idx, iters, mode in ((1, 10, "full"), (2, 2, "checkpointed")):
        data = synth.make(idx)
        cfg = data["cfg"]
        Zo, vo, oo = oracle.barycenter(data["Z0"], data["X"], data["offsets"], cfg.gamma, iters, cfg.step, mode=mode)
        Z = data["Z0"].astype(np.float64)
        hist = []
        for _ in range(iters):
            v, G, obj = oracle.value_grad_f64z(Z, data["X"], data["offsets"], cfg.gamma, mode=mode)
            hist.append(obj)
            Z = Z - cfg.step * G
        assert np.array_equal(Z, Zo) and np.array_equal(np.array(hist), oo) and np.array_equal(v, vo)
    # at a float32-representable Z it is value_grad itself
    data = synth.make(1)
    v1, g1, o1 = oracle.value_grad_f64z(data["Z0"].astype(np.float64), data["X"], data["offsets"], 1.0)
    v2, g2, o2 = oracle.value_grad(data["Z0"], data["X"], data["offsets"], 1.0, want_objective=True)
    assert np.array_equal(v1, v2) and np.array_equal(g1, g2) and o1 == o2


# ------------------------------------------------------------------------------------------- L-BFGS (Table 1; C23)
def _dense_bfgs_inverse(S, Y):
    """The inverse-Hessian approximation of BFGS after the pairs (s_i, y_i), oldest first, from H0 = (s.y / y.y of the
    newest pair) I, by the textbook update H <- (I - rho s y^T) H (I - rho y s^T) + rho s s^T, as a dense matrix."""
    n = S.shape[1]
    H = (S[-1] @ Y[-1]) / (Y[-1] @ Y[-1]) * np.eye(n)
    for s, y in zip(S, Y):
        rho = 1.0 / (s @ y)
        V = np.eye(n) - rho * np.outer(y, s)
        H = V.T @ H @ V + rho * np.outer(s, s)
    return H


def test_lbfgs_two_loop_recursion_is_the_dense_bfgs_operator(oracle):
    """oracle.lbfgs_direction (the two-loop recursion, Nocedal & Wright Alg. 7.4) against the dense BFGS matrix built by
    the update formula in numpy; the secant equation H y = s for the newest pair; no pairs = the identity."""
    rng = np.random.Generator(np.random.PCG64(555))
    n = 23
    A = rng.standard_normal((n, n))
    A = A @ A.T + n * np.eye(n)                              # curvature of a strictly convex quadratic: y = A s, s.y > 0
    for count in (1, 2, 5, 9):
        S = rng.standard_normal((count, n))
        Y = S @ A
        g = rng.standard_normal(n)
        r = oracle.lbfgs_direction(S, Y, g)
        H = _dense_bfgs_inverse(S, Y)
        assert np.abs(r - H @ g).max() <= 1e-12 * np.abs(H @ g).max()
        assert np.abs(oracle.lbfgs_direction(S, Y, Y[-1]) - S[-1]).max() <= 1e-12 * np.abs(S[-1]).max()   # secant equation
        # a transposed operand (y . q instead of s . q in the first loop) or swapped loop order breaks the symmetry of H
        g2 = rng.standard_normal(n)
        assert abs(g2 @ r - g @ oracle.lbfgs_direction(S, Y, g2)) <= 1e-10 * abs(g2 @ r)
    g = rng.standard_normal(n)
    assert np.array_equal(oracle.lbfgs_direction(np.zeros((0, n)), np.zeros((0, n)), g), g)


def test_lbfgs_descent_pins(oracle):
    """hist = 0 is the Armijo backtracking descent operation for operation; with history every accepted step satisfies
    the Armijo condition along its own direction (replayed with independent evaluations), the objective decreases
    monotonically, and after the first iteration the unit step is tried first."""
    data = synth.make(1)
    cfg = data["cfg"]
    Z0, X, off = data["Z0"], data["X"], data["offsets"]
    a = oracle.barycenter_backtracking(Z0, X, off, cfg.gamma, 6, 0.05)
    b = oracle.barycenter_lbfgs(Z0, X, off, cfg.gamma, 6, 0, 0.05)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    c1, step0 = 1e-4, 0.05
    # replay: drive the recursion here with independent evaluations (oracle.value_grad_f64z) and numpy vectors
    Z = Z0.astype(np.float64)
    Zl, vl, obj, steps, trials = oracle.barycenter_lbfgs(Z0, X, off, cfg.gamma, 7, 4, step0, 0.5, c1)
    assert np.all(np.diff(obj) < 0) and np.all(steps[1:] == 1.0) and steps[0] == step0
    S, Y = [], []
    v, G, f = oracle.value_grad_f64z(Z, X, off, cfg.gamma)
    for it in range(7):
        assert abs(f - obj[it]) <= 1e-12 * abs(f)
        d = -oracle.lbfgs_direction(np.array(S[-4:]), np.array(Y[-4:]), G.reshape(-1)).reshape(G.shape) if S else -G
        t = steps[it]
        Zn = Z + t * d
        vn, Gn, fn = oracle.value_grad_f64z(Zn, X, off, cfg.gamma)
        assert fn <= f + c1 * t * float((G * d).sum())                       # Armijo along the L-BFGS direction
        if trials[it] > 1:                                                   # the step before it was rejected
            tp = t / 0.5
            _, _, fp = oracle.value_grad_f64z(Z + tp * d, X, off, cfg.gamma, want_grad=False)
            assert fp > f + c1 * tp * float((G * d).sum())
        S.append((Zn - Z).reshape(-1)); Y.append((Gn - G).reshape(-1))
        Z, G, f = Zn, Gn, fn
    assert np.abs(Z - Zl).max() <= 1e-12 * np.abs(Zl).max() and abs(f - obj[7]) <= 1e-12 * abs(f)
    # L-BFGS beats plain backtracking descent on the same budget of iterations
    assert obj[7] < oracle.barycenter_backtracking(Z0, X, off, cfg.gamma, 7, step0, 0.5, c1)[2][7]
