"""GPU parity: the CUDA library (through its C ABI / thin binding) against the FP64 CPU oracle, element by element,
on identical seeded inputs.  Bars (BASELINE.json north_star):
  * neighbour counts / pair counts: bit-exact
  * V, rho, A: <= 4e-6 relative (max norm, 2x the measured worst);  B, grad A, grad B: <= 1e-4 relative L2 (normalised by rms)
  * dv/dt, du/dt: <= 1e-4 relative L2 (normalised by rms); conservation invariants <= 1e-5
Run with `pytest -m gpu` on a B200.
"""
import numpy as np
import pytest

import crk_workloads as wl

pytestmark = pytest.mark.gpu

TOL_DERIV = 1e-4
TOL_INV = 1e-5
TOL_WORST = 1e-3       # per particle: |dv/dt error| against the particle's own scale (check_parity)
TOL_SCALAR = 4e-6      # max-norm on V, rho, A.  Measured maxima over every case of this file (printed as [scalars]): V 1.3e-6,
                       # rho 1.3e-6 (n_h = 4, 268-term FP32 sums), A 1.8e-6 (non-default parameters); the bar is 2x the worst.
                       # Source: FP32 accumulation of 60-268 kernel terms, each through rsqrt.approx (2^-22) -- DESIGN.md 5.3


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return float(np.sqrt(((a - b) ** 2).sum() / max((b ** 2).sum(), 1e-300)))


def gpu_eval(ps, stages=False):
    """Evaluate the full path on the GPU through the binding; returns numpy arrays in caller order."""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    dev = torch.device("cuda:0")
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in
         ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")}
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h)
    ctx.build_cells(t["x"], t["y"], t["z"], t["h"])
    V, rho, cnt = ctx.volumes(t["m"])
    A, B, gA, gB = ctx.rk_coefficients()
    ax, ay, az, du, pc = ctx.hydro_derivs(t["vx"], t["vy"], t["vz"], t["u"])
    gv = ctx.gradv()
    perm = ctx.perm()
    torch.cuda.synchronize()
    out = dict(V=V, rho=rho, nbr_count=cnt, A=A, B=B, gradA=gA, gradB=gB, ax=ax, ay=ay, az=az, dudt=du,
               pair_count=pc, gradv=gv, perm=perm)
    out = {k: v.cpu().numpy() for k, v in out.items()}
    out["stats"] = ctx.stats()
    out["ctx"] = ctx
    return out


def check_parity(ps, g, o, oracle_gv=None, mask=None, label=""):
    """g: GPU outputs, o: oracle outputs (dicts).  mask: compare only these particles (windowed oracle)."""
    sel = slice(None) if mask is None else mask
    if mask is None and "stats" in g:     # both sides took the S14 branch (singular m2 -> B = 0 exactly) for the same number of particles
        assert g["stats"]["n_fallback"] == int((np.asarray(o["B"]) == 0.0).all(axis=0).sum()), label + " S14 fallback count"
    assert np.array_equal(g["nbr_count"][sel].astype(np.int64), o["nbr_count"][sel].astype(np.int64)), label + " nbr_count"
    assert np.array_equal(g["pair_count"][sel].astype(np.int64), o["pair_count"][sel].astype(np.int64)), label + " pair_count"
    e_s = [float(np.max(np.abs(g[k][sel] / o[k][sel] - 1))) for k in ("V", "rho", "A")]
    print(f"[scalars] {label}: max rel err V {e_s[0]:.2e} rho {e_s[1]:.2e} A {e_s[2]:.2e}")
    assert e_s[0] < TOL_SCALAR, label + " V"
    assert e_s[1] < TOL_SCALAR, label + " rho"
    assert e_s[2] < TOL_SCALAR, label + " A"
    for k in ("B", "gradA", "gradB"):
        e = rel_l2(g[k][:, sel], o[k][:, sel])
        assert e < TOL_DERIV, f"{label} {k} rel L2 {e:.3e}"
    if oracle_gv is not None:
        e = rel_l2(g["gradv"][:, sel], oracle_gv[:, sel])
        assert e < TOL_DERIV, f"{label} gradv rel L2 {e:.3e}"
    acc_g = np.stack([g["ax"][sel], g["ay"][sel], g["az"][sel]]); acc_o = np.stack([o["ax"][sel], o["ay"][sel], o["az"][sel]])
    e_a = rel_l2(acc_g, acc_o)
    e_u = rel_l2(g["dudt"][sel], o["dudt"][sel])
    assert e_a < TOL_DERIV, f"{label} dv/dt rel L2 {e_a:.3e}"
    assert e_u < TOL_DERIV, f"{label} du/dt rel L2 {e_u:.3e}"
    # a global norm is dominated by the particles with the largest derivatives (the cores of a clustered set): every particle
    # is also held to TOL_WORST of its OWN scale -- the larger of its acceleration and the pressure-gradient scale
    # (gamma - 1) u_i / h_i of a single pair term -- so that a wrong particle in a void cannot hide under the rms of the cores
    scale = np.maximum(np.sqrt((acc_o.astype(np.float64) ** 2).sum(0)),
                       (ps.gamma - 1.0) * np.abs(ps.u[sel].astype(np.float64)) / ps.h[sel].astype(np.float64))
    err = np.sqrt(((acc_g.astype(np.float64) - acc_o) ** 2).sum(0))
    worst = float((err / scale).max()) if err.size else 0.0
    print(f"[worst particle] {label}: |dv/dt error| / max(|dv/dt|, (gamma-1) u/h) = {worst:.2e}")
    assert worst < TOL_WORST, f"{label} worst particle {worst:.3e}"
    return e_a, e_u


def check_invariants(ps, g, label=""):
    m = ps.m.astype(np.float64)
    a = [g[k].astype(np.float64) for k in ("ax", "ay", "az")]
    v = [ps.vx.astype(np.float64), ps.vy.astype(np.float64), ps.vz.astype(np.float64)]
    mom = max(abs((m * a[q]).sum()) for q in range(3)) / (m * np.sqrt(a[0] ** 2 + a[1] ** 2 + a[2] ** 2)).sum()
    du = g["dudt"].astype(np.float64)
    work = m * (v[0] * a[0] + v[1] * a[1] + v[2] * a[2])
    en = abs((work + m * du).sum()) / ((m * np.abs(du)).sum() + np.abs(work).sum() + 1e-300)
    assert mom < TOL_INV, f"{label} momentum residual {mom:.3e}"
    assert en < TOL_INV, f"{label} energy residual {en:.3e}"
    return mom, en


# ------------------------------------------------------------------------------------------------ structure
def test_sort_tree_and_leaf_lists_cover_every_neighbour(oracle_mod):
    ps = wl.clustered_plummer(n_side=20)
    g = gpu_eval(ps)
    n = ps.n
    perm = g["perm"].astype(np.int64)
    assert np.array_equal(np.sort(perm), np.arange(n)), "perm is not a permutation"
    slot = np.empty(n, dtype=np.int64); slot[perm] = np.arange(n)
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
    o.build(ps.x, ps.y, ps.z, ps.h)
    ctx = g["ctx"]
    st = g["stats"]
    assert st["n_leaves"] == (n + 31) // 32
    rng = np.random.default_rng(0)
    for leaf in rng.integers(0, st["n_leaves"], 60):
        lst = ctx.leaf_list(int(leaf))
        ids = (lst & np.uint32(0x0fffffff)).astype(np.int64)
        assert np.all(np.diff(ids) > 0), "leaf list not strictly ascending"
        gather = set(ids[(lst >> np.uint32(31)) == 1].tolist()); allb = set(ids.tolist())
        for k in range(leaf * 32, min(leaf * 32 + 32, n)):
            js, fi, fj = o.neighbors(perm[k])
            lj = slot[js.astype(np.int64)] // 32
            assert set(lj.tolist()) <= allb, "a symmetric neighbour's leaf is missing from the list"
            assert set(lj[fi].tolist()) <= gather, "a gather neighbour's leaf lacks the gather flag"


def test_joint_tree_walk_builds_the_lists_of_the_per_leaf_walk():
    """cosmo 128^3 = 2048 level-1 nodes of similar supports: crk_build_cells walks the tree once per node of 32 leaves; with
    CRK_FLAG_TREE_PER_LEAF once per leaf.  Same entries, same order, same flags -- and so the same bits downstream."""
    import torch
    from paper_2202_02840_b200 import Crk
    ps = wl.make_config("cosmo", 128)
    dev = torch.device("cuda:0")
    t = [torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")]
    outs = []
    lists = []
    for per_leaf in (False, True):
        ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h, tree_per_leaf=per_leaf)
        out = ctx.step_derivs(*t)
        torch.cuda.synchronize()
        st = ctx.stats()
        rng = np.random.default_rng(1)
        lists.append((st["n_leaf_pairs"], st["n_leaf_pairs_gather"], [ctx.leaf_list(int(q)) for q in rng.integers(0, st["n_leaves"], 200)]))
        outs.append([o.cpu().numpy() for o in out])
    assert lists[0][0] == lists[1][0] and lists[0][1] == lists[1][1], "leaf pair totals differ"
    for a, b in zip(lists[0][2], lists[1][2]):
        assert np.array_equal(a, b), "a leaf interaction list differs between the two walks"
    for a, b in zip(outs[0], outs[1]):
        assert np.array_equal(a.view(np.uint32), b.view(np.uint32)), "derivatives differ in some bit"


# ------------------------------------------------------------------------------------------------ small configs
@pytest.mark.parametrize("name,n_side", [("tiny_uniform", 16), ("blast_wave", 24), ("clustered", 24), ("cosmo", 32)])
def test_parity_small(name, n_side, oracle_mod):
    ps = wl.make_config(name, n_side)
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
    od = o.step_derivs(ps)
    g = gpu_eval(ps)
    e_a, e_u = check_parity(ps, g, od, oracle_gv=o.gradv(), label=name)
    mom, en = check_invariants(ps, g, label=name)
    print(f"[parity] {name} n={ps.n}: dv/dt {e_a:.2e} du/dt {e_u:.2e} momentum {mom:.2e} energy {en:.2e}")


def test_parity_ragged_sizes(oracle_mod):
    """N not a multiple of the 32-particle leaf, including a single leaf and a single particle"""
    base = wl.tiny_uniform(n_side=10)
    for n in (1, 2, 31, 33, 257, 999):
        ps = base.subset(np.arange(n))
        ps.h = np.full(n, 0.2, np.float32)
        o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
        od = o.step_derivs(ps)
        g = gpu_eval(ps)
        assert np.array_equal(g["nbr_count"].astype(np.int64), od["nbr_count"].astype(np.int64))
        assert np.array_equal(g["pair_count"].astype(np.int64), od["pair_count"].astype(np.int64))
        assert np.max(np.abs(g["V"] / od["V"] - 1)) < TOL_SCALAR
        if n >= 257:
            check_parity(ps, g, od, label=f"ragged{n}")


def test_parity_coincident_particles(oracle_mod):
    """S14: exact duplicates (r = 0, i != j), which FP32 rounding produces in Plummer cores.  Every formula is finite there
    (D = W'/r carries no 1/r, mu = 0, phi_ad = exp(-25)); the pair is a neighbour and is counted."""
    ps = wl.tiny_uniform(n_side=12, seed=31)
    rng = np.random.default_rng(3)
    src = rng.choice(ps.n, 80, replace=False)
    dst = src[:40]; ref = src[40:]
    for k in ("x", "y", "z"):
        a = getattr(ps, k); a[dst] = a[ref]
    # three particles on one point as well
    for k in ("x", "y", "z"):
        a = getattr(ps, k); a[dst[0]] = a[ref[1]]
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
    od = o.step_derivs(ps)
    g = gpu_eval(ps)
    e_a, e_u = check_parity(ps, g, od, oracle_gv=o.gradv(), label="coincident")
    check_invariants(ps, g, label="coincident")
    assert all(np.isfinite(g[k]).all() for k in ("ax", "ay", "az", "dudt", "A", "B", "gradA", "gradB", "gradv"))
    print(f"[parity] coincident particles: dv/dt {e_a:.2e} du/dt {e_u:.2e}")


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_parity_singular_m2_fallback(n, oracle_mod):
    """S14: n = 1, 2, 3 particles (and 4 coplanar ones) cannot span three dimensions, m2 is singular and both sides must take
    the zeroth-order correction B = 0, grad B = 0, A = 1/m0, grad A = -A^2 grad m0; every output is compared."""
    pts = np.array([[0.50, 0.50, 0.50], [0.55, 0.52, 0.49], [0.47, 0.56, 0.53], [0.53, 0.58, 0.52]])[:n]
    if n == 4:                                   # make the fourth point coplanar with the first three
        pts[3] = pts[0] + 0.7 * (pts[1] - pts[0]) - 0.4 * (pts[2] - pts[0])
    base = wl.tiny_uniform(n_side=4)
    ps = base.subset(np.arange(n))
    ps.x, ps.y, ps.z = (pts[:, q].astype(np.float32) for q in range(3))
    ps.h = np.full(n, 0.2, np.float32)
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
    od = o.step_derivs(ps)
    g = gpu_eval(ps)
    assert np.abs(od["B"]).max() == 0.0 and np.abs(od["gradB"]).max() == 0.0, "the oracle did not take the S14 branch"
    assert np.abs(g["B"]).max() == 0.0 and np.abs(g["gradB"]).max() == 0.0, "the kernel did not take the S14 branch"
    assert g["stats"]["n_fallback"] == n, "crk_stats.n_fallback counts the particles that took it"
    assert np.array_equal(g["nbr_count"].astype(np.int64), od["nbr_count"].astype(np.int64))
    assert np.array_equal(g["pair_count"].astype(np.int64), od["pair_count"].astype(np.int64))
    assert np.allclose(g["V"], od["V"], rtol=TOL_SCALAR) and np.allclose(g["A"], od["A"], rtol=TOL_SCALAR)
    sA = np.abs(od["gradA"]).max()
    assert np.abs(g["gradA"] - od["gradA"]).max() <= 1e-4 * sA + 1e-30
    gv = o.gradv()
    assert np.abs(g["gradv"] - gv).max() <= 1e-4 * np.abs(gv).max() + 1e-30
    for k in ("ax", "ay", "az", "dudt"):
        sc = max(np.abs(od[k]).max(), 1e-30)
        assert np.abs(g[k] - od[k]).max() <= 1e-4 * sc, k


def test_parity_on_both_sides_of_the_singularity_line(oracle_mod):
    """S14 near its threshold: a disc of 20 particles walked off its plane, as in tests/test_oracle_pins.py.  The oracle forms
    det m2 / (tr m2 / 3)^3 from FP64 sums, the library from FP32 sums, so a particle within rounding of 1e-4 may
    legitimately take different branches; every set here keeps all its particles at least a factor 1.25 away from the line
    (sets that do not are passed over, and at least three on each side must remain).  Then both sides must take the same
    branch for every particle (crk_stats.n_fallback and the pattern of B = 0 against the oracle's ratios), counts and
    volumes must agree as everywhere, and the sets that are entirely in the fallback (well-conditioned: A = 1/m0) meet every
    bar of check_parity.  Above the line the condition number of m2 grows like 4 / ratio (printed as "growth"); the errors of
    B and dv/dt are reported per set and held to the usual 1e-4 (measured on a B200: <= 3e-7 down to a ratio of 1.7e-4 --
    the eta-normalised FP32 sums lose nothing there that the FP64 solve would amplify)."""
    rng = np.random.default_rng(1405)
    disc = 0.09 * rng.uniform(-1, 1, (20, 2))
    xi = rng.uniform(-1, 1, 20)
    base = wl.tiny_uniform(n_side=4)
    used = {"all_fallback": 0, "none_fallback": 0, "mixed": 0}
    for eps in np.logspace(-3.5, -1.0, 26):
        pts = np.array([0.5, 0.5, 0.5]) + np.c_[disc, 0.09 * eps * xi]
        ps = base.subset(np.arange(20))
        ps.x, ps.y, ps.z = (pts[:, q].astype(np.float32) for q in range(3))
        ps.h = np.full(20, 0.2, np.float32)
        o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
        od = o.step_derivs(ps)
        m0, m1, m2 = o.moments()
        M = m2.T.reshape(-1, 3, 3)
        ratio = np.linalg.det(M) / (np.trace(M, axis1=1, axis2=2) / 3.0) ** 3
        if np.any((ratio > 0.8e-4) & (ratio < 1.25e-4)):
            continue
        g = gpu_eval(ps)
        nfb = int((ratio <= 1e-4).sum())
        assert g["stats"]["n_fallback"] == nfb, f"eps {eps:.2e}: library {g['stats']['n_fallback']} fallbacks, oracle {nfb}"
        assert np.array_equal((g["B"] == 0).all(axis=0), ratio <= 1e-4)
        assert np.array_equal(g["nbr_count"].astype(np.int64), od["nbr_count"].astype(np.int64))
        assert np.array_equal(g["pair_count"].astype(np.int64), od["pair_count"].astype(np.int64))
        assert np.abs(g["V"] / od["V"] - 1).max() < TOL_SCALAR
        if nfb == 20:
            check_parity(ps, g, od, oracle_gv=o.gradv(), label=f"disc eps={eps:.1e} (all in the fallback)")
        else:
            e_B = rel_l2(g["B"], od["B"])
            e_a = rel_l2(np.stack([g["ax"], g["ay"], g["az"]]), np.stack([od["ax"], od["ay"], od["az"]]))
            grow = 4.0 / float(ratio[ratio > 1e-4].min())
            print(f"[S14] disc eps={eps:.1e}: {nfb} of 20 in the fallback, smallest ratio above the line {ratio[ratio > 1e-4].min():.2e}: "
                  f"B rel L2 {e_B:.2e}, dv/dt rel L2 {e_a:.2e} (condition growth ~{grow:.0f}x)")
            assert e_B < TOL_DERIV and e_a < TOL_DERIV
        used["all_fallback" if nfb == 20 else ("none_fallback" if nfb == 0 else "mixed")] += 1
    print(f"[S14] sets compared: {used}")
    assert used["all_fallback"] >= 3 and used["none_fallback"] >= 3


def test_parity_negative_internal_energy(oracle_mod):
    """S12: u < 0 on some particles (forward Euler with Eq. 18 drives cold shell particles there): P = (gamma-1) rho u stays
    unclamped (negative), c_s uses max(u, 0); entropy <= 0 makes the compatible partition f_ij = 1/2 (S16)."""
    ps = wl.tiny_uniform(n_side=14, seed=41)
    rng = np.random.default_rng(5)
    neg = rng.choice(ps.n, ps.n // 10, replace=False)
    ps.u[neg] = -ps.u[neg] * np.float32(0.3)
    ps.u[neg[:20]] = 0.0
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
    od = o.step_derivs(ps)
    g = gpu_eval(ps)
    e_a, e_u = check_parity(ps, g, od, oracle_gv=o.gradv(), label="u<0")
    check_invariants(ps, g, label="u<0")
    torch = _torch()
    du = g["ctx"].compatible_energy(1e-3).cpu().numpy()
    e_c = rel_l2(du, o.compatible_energy(1e-3))
    assert e_c < TOL_DERIV
    print(f"[parity] u<0 on {len(neg)} particles: dv/dt {e_a:.2e} du/dt {e_u:.2e} compatible du {e_c:.2e}")


@pytest.mark.parametrize("name,n_side,frac", [("clustered", 24, 0.10), ("cosmo", 32, 0.25), ("tiny_uniform", 16, 1.0)])
def test_active_particles_parity(name, n_side, frac, oracle_mod):
    """NEXT row 4b: derivatives of the active particles only.  Active = the `frac` of the particles with the
    smallest h (the ones a hierarchical time-step scheme would put in the deepest bins); compared with the oracle's
    restricted sums, with the library's own full evaluation (same kernels, so identical bits), and passive entries stay
    untouched."""
    torch = _torch()
    ps = wl.make_config(name, n_side)
    order = np.argsort(ps.h, kind="stable")
    active = np.zeros(ps.n, dtype=np.uint8)
    active[order[:max(1, int(frac * ps.n))]] = 1
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
    o.step_derivs(ps)
    oa = o.hydro_derivs_active(active, ps.vx, ps.vy, ps.vz, ps.u)
    g = gpu_eval(ps)
    ctx = g["ctx"]
    dev = torch.device("cuda:0")
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in ("vx", "vy", "vz", "u")}
    # velocities changed since the last full evaluation: the active call must redo grad v of the halo leaves
    ctx.hydro_derivs(t["vx"] * 0.5, t["vy"] * 0.5, t["vz"] * 0.5, t["u"])
    out = ctx.hydro_derivs_active(torch.from_numpy(active).to(dev), t["vx"], t["vy"], t["vz"], t["u"])
    torch.cuda.synchronize()
    st = ctx.stats()
    on = active != 0
    got = [q.cpu().numpy() for q in out]
    for q, k in zip(got, ("ax", "ay", "az", "dudt")):
        assert np.isnan(q[~on]).all(), "a passive entry was written"
        assert np.array_equal(q[on], g[k][on]), "active results differ from the full evaluation"
    e_a = rel_l2(np.stack([q[on] for q in got[:3]]), np.stack([q[on] for q in oa[:3]]))
    e_u = rel_l2(got[3][on], oa[3][on])
    assert e_a < TOL_DERIV and e_u < TOL_DERIV
    assert 0 < st["n_active_leaves"] <= st["n_leaves"] and st["n_active_leaves"] <= st["n_halo_leaves"] <= st["n_leaves"]
    if frac == 1.0:
        assert st["n_active_leaves"] == st["n_leaves"]
    print(f"[active] {name}: {on.sum()} of {ps.n} particles active, leaves active {st['n_active_leaves']} halo {st['n_halo_leaves']} "
          f"of {st['n_leaves']}; dv/dt {e_a:.2e} du/dt {e_u:.2e}")


def test_kdk_reuse_is_dropped_when_h_evolves():
    """CRK_FLAG_KDK_REUSE keeps lists, volumes and coefficients between consecutive crk_kdk_step calls on the same arrays;
    crk_evolve_h followed by an in-place change of h (the integration loop of the Sod / Sedov tests) must drop that reuse."""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    ps = wl.tiny_uniform()
    dev = torch.device("cuda:0")
    names = ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")

    def run(reuse):
        t = [torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in names]
        ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h, kdk_reuse=reuse)
        for _ in range(3):
            ctx.kdk_step(*t, 2e-3)
            t[3].copy_(ctx.evolve_h() * 1.05)          # same address, new values
        torch.cuda.synchronize()
        return [q.cpu().numpy() for q in t]

    a, b = run(False), run(True)
    for qa, qb, k in zip(a, b, names):
        assert np.array_equal(qa, qb), k


def test_build_does_not_depend_on_the_history_of_the_context():
    """crk_build_cells runs on the key width, leaf-list capacity and arena size the previous build found and synchronises once;
    if the new data outgrew one of them the build is repeated.  A context that has seen other data must give the bits of a
    fresh one (different smallest h -> different key width; denser lists -> larger capacity / arena)."""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    dev = torch.device("cuda:0")
    names = ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")
    sets = [wl.tiny_uniform(), wl.clustered_plummer(n_side=20), wl.zeldovich(n_side=24), wl.tiny_uniform(n_side=10)]
    sets[3].h = (sets[3].h * np.float32(1.6)).astype(np.float32)          # 4x the neighbours, lists outgrow the first guess

    def evaluate(ctx, ps):
        t = [torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in names]
        out = ctx.step_derivs(*t)
        torch.cuda.synchronize()
        return [o.cpu().numpy() for o in out]

    fresh = [evaluate(Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h), ps) for ps in sets]
    used = Crk(box=sets[0].box, gamma=sets[0].gamma, n_h=sets[0].n_h)
    for order in ((0, 1, 2, 3), (3, 2, 1, 0), (1, 1, 3, 0)):
        for k in order:
            got = evaluate(used, sets[k])
            for a, b in zip(got, fresh[k]):
                assert np.array_equal(a, b), f"set {k} after other data differs from a fresh context"
    assert used.stats()["rebuilds"] >= 1


def test_step_derivs_and_host_entry_match_staged_calls():
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    ps = wl.tiny_uniform()
    g = gpu_eval(ps)
    dev = torch.device("cuda:0")
    names = ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")
    t = [torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in names]
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h)
    out = ctx.step_derivs(*t)
    torch.cuda.synchronize()
    for o, k in zip(out, ("ax", "ay", "az", "dudt")):
        assert np.array_equal(o.cpu().numpy(), g[k]), k
    th = [torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).pin_memory() for k in names]
    oh = [torch.empty(ps.n).pin_memory() for _ in range(4)]
    ctx.step_derivs_host(*th, oh)
    for o, k in zip(oh, ("ax", "ay", "az", "dudt")):
        assert np.array_equal(o.numpy(), g[k]), k
    # determinism: a second evaluation gives identical bits
    out2 = ctx.step_derivs(*t)
    torch.cuda.synchronize()
    for a, b in zip(out, out2):
        assert torch.equal(a, b)


def test_errors_and_empty_input():
    torch = _torch()
    from paper_2202_02840_b200 import Crk, CrkError
    dev = torch.device("cuda:0")
    ctx = Crk()
    e = torch.empty(0, device=dev)
    out = ctx.step_derivs(e, e, e, e, e, e, e, e, e)
    assert all(o.numel() == 0 for o in out)
    one = torch.full((4,), 0.5, device=dev)
    with pytest.raises(CrkError) as ei:
        ctx.build_cells(one, one, one, torch.full((4,), 0.5, device=dev))       # h >= L/2
    assert ei.value.code == -2
    with pytest.raises(CrkError) as ei:
        ctx.build_cells(torch.full((4,), 1.0, device=dev), one, one, torch.full((4,), 0.1, device=dev))
    assert ei.value.code == -2
    ctx2 = Crk()
    with pytest.raises(CrkError) as ei:
        ctx2.volumes(one)
    assert ei.value.code == -5
    ctx2.build_cells(torch.rand(4, device=dev), torch.rand(4, device=dev), torch.rand(4, device=dev),
                     torch.full((4,), 0.1, device=dev))
    with pytest.raises(CrkError) as ei:
        ctx2.hydro_derivs(one, one, one, one)
    assert ei.value.code == -5
    # next rows: wrong call order / missing flag -> CRK_ESTATE; empty input is fine; a step that leaves the box is caught
    for call in (lambda: ctx2.evolve_h(), lambda: ctx2.compatible_energy(1e-3), lambda: ctx2.timestep(0.25)):
        with pytest.raises(CrkError) as ei:
            call()
        assert ei.value.code == -5
    ctx3 = Crk(timestep=True, kdk_compatible=True, kdk_reuse=True)
    ctx3.kdk_step(e, e, e, e, e, e, e, e, e, 1e-3)
    r = lambda: torch.rand(64, device=dev)
    st = [r(), r(), r(), torch.full((64,), 0.2, device=dev), r(), r(), r(), torch.full((64,), 1.0 / 64, device=dev), r() + 1.0]
    ctx3.kdk_step(*st, 1e-3)
    assert all(torch.isfinite(q).all() for q in st)
    st[4].fill_(float("nan"))                                                  # v = NaN -> positions leave [0, L)
    with pytest.raises(CrkError) as ei:
        ctx3.kdk_step(*st, 1e-3)
        ctx3.kdk_step(*st, 1e-3)
    assert ei.value.code == -2


# ------------------------------------------------------------------------------------------------ config 2 multi-step
def test_blast_wave_teacher_forced_euler_steps(oracle_mod):
    """Config 2's protocol at reduced size and step, against the O(N^2) brute-force build (the full-size, full-dt protocol
    is test_config2_protocol_as_written): at each Euler step the GPU evaluates derivatives on the oracle's FP32 state
    and must meet the bar; states come from oracle/crk_oracle.py:euler_steps (FP64 update)."""
    ps = wl.blast_wave(n_side=24)
    worst = 0.0
    for step, cur, od in oracle_mod.euler_steps(ps, 6, 1e-4 * (64 / 24) ** 0 * 0.25):
        g = gpu_eval(cur)
        e_a, e_u = check_parity(cur, g, od, label=f"blast step {step}")
        worst = max(worst, e_a, e_u)
    print(f"[parity] blast teacher-forced worst rel L2 {worst:.2e}")


def _gpu_euler_free_run(ps, n_steps, dt):
    """forward Euler on the GPU's own FP32 state: three AXPYs on the caller's tensors around crk_step_derivs (the update
    rule of DESIGN.md step 12 / S12; kept in the test, the library only evaluates derivatives).  Yields (step, state, derivs)."""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    dev = torch.device("cuda:0")
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in
         ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")}
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h)
    L = float(ps.box)
    for step in range(n_steps + 1):
        out = ctx.step_derivs(*[t[k] for k in ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")])
        torch.cuda.synchronize()
        yield step, {k: v.cpu().numpy() for k, v in t.items()}, [o.cpu().numpy() for o in out]
        if step == n_steps:
            break
        for xk, vk, a in (("x", "vx", out[0]), ("y", "vy", out[1]), ("z", "vz", out[2])):
            p = t[xk] + t[vk] * dt
            p = p - torch.floor(p / L) * L
            p[(p >= L) | (p < 0)] = 0.0
            t[xk] = p
            t[vk] = t[vk] + a * dt
        t["u"] = t["u"] + out[3] * dt


def test_config2_protocol_as_written(oracle_mod):
    """BASELINE.json configs[1] at its stated size and step: 64^3 blast wave, one derivative evaluation plus 10 forward-Euler
    steps at fixed dt = 1e-4 (4.9x the CFL step of the hot centre: the trajectory explodes from step ~6, reading S12).
    (ii) teacher-forced: at every state of the oracle's FP64 trajectory the GPU evaluates the derivatives of the FP32 cast of
         that state and must meet the bars (counts bit-exact, 1e-4 rel L2), as long as the oracle's values fit FP32;
    (iii) free-running GPU trajectory against the oracle's, reported per step with the step at which it leaves 1e-4."""
    ps = wl.blast_wave()
    dt = 1e-4
    assert ps.n == 64 ** 3
    fp32_ok = 1e30        # beyond this the derivatives leave the range in which FP32 products are safe (3.4e38)
    oracle_states = []
    worst, asserted = 0.0, 0
    for step, cur, od in oracle_mod.euler_steps(ps, 10, dt, grid=True):
        big = max(np.abs(od["dudt"]).max(), np.abs(od["ax"]).max(), np.abs(od["ay"]).max(), np.abs(od["az"]).max())
        oracle_states.append((cur, od))
        g = gpu_eval(cur)
        if big < fp32_ok:
            e_a, e_u = check_parity(cur, g, od, label=f"config2 teacher-forced state {step}")
            worst = max(worst, e_a, e_u)
            asserted += 1
            print(f"[config2 dt=1e-4] teacher-forced state {step}: dv/dt {e_a:.2e} du/dt {e_u:.2e} (max |deriv| {big:.1e}, u<0: {(cur.u < 0).sum()})")
        else:
            fin = all(np.isfinite(g[k]).all() for k in ("ax", "ay", "az", "dudt"))
            assert np.array_equal(g["nbr_count"].astype(np.int64), od["nbr_count"].astype(np.int64))
            assert np.array_equal(g["pair_count"].astype(np.int64), od["pair_count"].astype(np.int64))
            print(f"[config2 dt=1e-4] teacher-forced state {step}: oracle max |deriv| {big:.1e} is outside the FP32-safe range; "
                  f"GPU output finite: {fin}; counts bit-exact (reported, not asserted: S12)")
    assert asserted >= 9 and worst < TOL_DERIV
    left = None
    for (step, st, d), (cur, od) in zip(_gpu_euler_free_run(ps, 10, dt), oracle_states):
        with np.errstate(all="ignore"):
            e_v = rel_l2(np.stack([st["vx"], st["vy"], st["vz"]]), np.stack([cur.vx, cur.vy, cur.vz])) if step else 0.0
            e_a = rel_l2(np.stack(d[:3]), np.stack([od["ax"], od["ay"], od["az"]]))
            e_u = rel_l2(d[3], od["dudt"])
        if left is None and not (max(e_a, e_u) < TOL_DERIV):
            left = step
        print(f"[config2 dt=1e-4] free-running step {step}: state v {e_v:.2e}, dv/dt {e_a:.2e}, du/dt {e_u:.2e}")
    print(f"[config2 dt=1e-4] free-running GPU trajectory leaves the 1e-4 bar at step {left} (reported, not asserted)")


def test_config2_stable_variant_free_running(oracle_mod):
    """Labelled NON-BASELINE variant of config 2 (S12 iv): the same 64^3 blast wave at dt = 2e-5 (1x the CFL step), where a
    free-running comparison is meaningful: 10 forward-Euler steps on the GPU's own FP32 state against the oracle's FP64
    trajectory; derivatives at every step within 1e-4 rel L2, velocities and energies of the state within 1e-5."""
    ps = wl.blast_wave()
    dt = 2e-5
    worst_d, worst_s = 0.0, 0.0
    for (step, st, d), (_, cur, od) in zip(_gpu_euler_free_run(ps, 10, dt), oracle_mod.euler_steps(ps, 10, dt, grid=True)):
        e_a = rel_l2(np.stack(d[:3]), np.stack([od["ax"], od["ay"], od["az"]]))
        e_u = rel_l2(d[3], od["dudt"])
        e_v = rel_l2(np.stack([st["vx"], st["vy"], st["vz"]]), np.stack([cur.vx, cur.vy, cur.vz])) if step else 0.0
        e_e = rel_l2(st["u"], cur.u)
        dx = np.abs(st["x"].astype(np.float64) - cur.x.astype(np.float64))
        dx = np.minimum(dx, ps.box - dx).max()
        print(f"[config2 dt=2e-5] free-running step {step}: dv/dt {e_a:.2e} du/dt {e_u:.2e} | state v {e_v:.2e} u {e_e:.2e} x {dx:.1e}")
        worst_d = max(worst_d, e_a, e_u)
        worst_s = max(worst_s, e_v, e_e)
        assert dx < 1e-6
    assert worst_d < TOL_DERIV and worst_s < 1e-5


# ------------------------------------------------------------------------------------------------ BASELINE sizes
def _pick_window(ps, c, half, cap=120000):
    """Padded window such that every quantity of the core particles is determined inside it: hop 1 = symmetric set
    (r < max(h_i,h_j): a far particle with a large h_j can reach the core), hops 2-3 = gather sets of radius <= hmax."""
    cc = np.asarray(c, dtype=np.float64)
    off = np.zeros(ps.n)
    for a_, k in enumerate(("x", "y", "z")):
        d = getattr(ps, k).astype(np.float64) - cc[a_]
        d -= np.round(d)
        off = np.maximum(off, np.abs(d))
    dist = np.maximum(off - half, 0.0)                     # Chebyshev distance to the core box (<= Euclidean)
    h = ps.h.astype(np.float64)
    core = off <= half
    if not core.any():
        return None
    hc = h[core].max()
    partners = dist < np.maximum(h, hc)                    # superset of the hop-1 partners of the core
    r1 = dist[partners].max()
    pad = r1 + 2.0 * h[partners].max()
    for _ in range(8):
        inside = off <= half + pad
        need = r1 + 2.0 * h[inside & (dist <= r1 + h[inside].max())].max()
        if need <= pad * (1 + 1e-9):
            break
        pad = need
    inside = off <= half + pad
    if inside.sum() > cap:
        return None
    idx = np.nonzero(inside)[0]
    return idx, core[idx]


def _window_check(ps, oracle_mod, centres, half_in_h=2.5, label=""):
    """windowed brute force: the oracle gets every particle of a padded window; only
    the un-padded core is compared."""
    g = gpu_eval(ps)
    check_invariants(ps, g, label=label)
    done = 0
    for c in centres:
        idx0, _ = wl.select_window(ps, c, 0.03, 0.0)
        if len(idx0) == 0:
            continue
        half = half_in_h * float(np.median(ps.h[idx0]))
        win = _pick_window(ps, c, half)
        if win is None:
            print(f"[parity] {label} window@{np.round(c, 3)} skipped (too many particles in the padded window)")
            continue
        idxp, corep = win
        sub = ps.subset(idxp)
        o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
        od = o.step_derivs(sub)
        gs = {k: (v[idxp] if v.ndim == 1 else v[:, idxp]) for k, v in g.items() if isinstance(v, np.ndarray) and k != "perm"}
        e_a, e_u = check_parity(sub, gs, od, oracle_gv=o.gradv(), mask=corep, label=f"{label} window@{np.round(c, 3)}")
        print(f"[parity] {label} window n={len(idxp)} core={int(corep.sum())}: dv/dt {e_a:.2e} du/dt {e_u:.2e}")
        done += 1
    assert done >= 1
    return g


def _full_count_check(ps, g, oracle_mod, label):
    """bit-exact neighbour / pair counts of EVERY particle against the oracle's grid formulation (oracle at scale)"""
    cg, cs = oracle_mod.grid_counts(ps)
    assert np.array_equal(np.asarray(g["nbr_count"]).astype(np.uint32), cg), label + " nbr_count (all particles)"
    assert np.array_equal(np.asarray(g["pair_count"]).astype(np.uint32), cs), label + " pair_count (all particles)"
    print(f"[parity] {label}: counts of all {ps.n} particles bit-exact (gather {int(cg.sum())}, symmetric {int(cs.sum())})")


def test_parity_config2_blast_full(oracle_mod):
    ps = wl.make_config("blast_wave")
    c = [(0.5, 0.5, 0.5), (0.1, 0.9, 0.3)]
    g = _window_check(ps, oracle_mod, c, half_in_h=3.0, label="blast64")
    _full_count_check(ps, g, oracle_mod, "blast64")


def test_parity_config3_clustered_full(oracle_mod):
    ps = wl.make_config("clustered")
    rng = np.random.default_rng(1)
    dens = np.argsort(ps.h)[:3]                      # densest cores
    centres = [(float(ps.x[i]), float(ps.y[i]), float(ps.z[i])) for i in dens] + [tuple(rng.random(3)) for _ in range(3)]
    _window_check(ps, oracle_mod, centres, half_in_h=2.0, label="clustered128")


def test_parity_config4_cosmo_full(oracle_mod):
    ps = wl.make_config("cosmo")
    centres = [(0.5, 0.5, 0.5), (0.001, 0.999, 0.5), (0.25, 0.75, 0.1)]
    g = _window_check(ps, oracle_mod, centres, half_in_h=3.0, label="cosmo256")
    _full_count_check(ps, g, oracle_mod, "cosmo256")
    st = g["stats"]
    print(f"[stats] cosmo256 leaves={st['n_leaves']} leaf_pairs={st['n_leaf_pairs']} launches={st['launches']}")
    # NEXT row 1 at the full size: the exactness property of PAPER.md:141 holds at any size
    torch = _torch()
    dt = 1e-2
    du = g["ctx"].compatible_energy(dt)
    torch.cuda.synchronize()
    du = du.cpu().numpy().astype(np.float64)
    m = ps.m.astype(np.float64)
    v = np.stack([ps.vx, ps.vy, ps.vz]).astype(np.float64)
    a = np.stack([g["ax"], g["ay"], g["az"]]).astype(np.float64)
    dke = 0.5 * (m * (((v + a * dt) ** 2).sum(0) - (v ** 2).sum(0))).sum()
    res = abs(dke + (m * du).sum()) / (m * np.abs(du)).sum()
    assert res < TOL_INV, f"cosmo256 compatible energy residual {res:.3e}"
    print(f"[parity] cosmo256 compatible energy residual {res:.2e}")


def _large_config_check(ps, oracle_mod, label, full_counts):
    """A 512^3 configuration through the staged API.  The full outputs stay on the GPU (invariants are reduced there in FP64);
    only the padded oracle windows come back.  Reports what BASELINE.json says about the config: h range, neighbour numbers,
    multi-segment leaves, and the time of every pass (first call, allocation included)."""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    dev = torch.device("cuda:0")
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in
         ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")}
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h)
    ctx.set_timing(True)
    ctx.build_cells(t["x"], t["y"], t["z"], t["h"])
    V, rho, cnt = ctx.volumes(t["m"])
    A, B, gA, gB = ctx.rk_coefficients()
    ax, ay, az, du, pc = ctx.hydro_derivs(t["vx"], t["vy"], t["vz"], t["u"])
    gv = ctx.gradv()
    torch.cuda.synchronize()
    st = ctx.stats()
    seg = ctx.leaf_segments().cpu().numpy().astype(np.uint32)
    print(f"[stats] {label} n={ps.n} leaves={st['n_leaves']} leaf_pairs={st['n_leaf_pairs']} ms: sort {st['ms_sort']:.1f} "
          f"tree {st['ms_tree']:.1f} lists {st['ms_lists']:.1f} volumes {st['ms_volumes']:.1f} rk {st['ms_rk']:.1f} "
          f"gradv {st['ms_gradv']:.1f} forces {st['ms_forces']:.1f}; gather neighbours mean "
          f"{float(cnt.to(torch.float64).mean()):.1f} max {int(cnt.max())}, pairs mean {float(pc.to(torch.float64).mean()):.1f} "
          f"max {int(pc.max())}; h max/min {float(ps.h.max() / ps.h.min()):.1f}, p99/p1 "
          f"{float(np.percentile(ps.h, 99) / np.percentile(ps.h, 1)):.1f}; multi-segment leaves {float((seg[:, 0] != 0).mean()):.3f}; "
          f"lists {st['list_bytes'] / 1e9:.1f} GB, scratch {st['scratch_bytes'] / 1e9:.1f} GB, rebuilds {st['rebuilds']}")
    # conservation invariants on the full output, FP64 on the device
    m = t["m"].double()
    a3 = [q.double() for q in (ax, ay, az)]
    v3 = [t[k].double() for k in ("vx", "vy", "vz")]
    amag = torch.sqrt(a3[0] ** 2 + a3[1] ** 2 + a3[2] ** 2)
    mom = max(abs(float((m * a3[q]).sum())) for q in range(3)) / float((m * amag).sum())
    work = m * (v3[0] * a3[0] + v3[1] * a3[1] + v3[2] * a3[2])
    en = abs(float((work + m * du.double()).sum())) / (float((m * du.double().abs()).sum()) + float(work.abs().sum()))
    assert mom < TOL_INV and en < TOL_INV, (mom, en)
    del m, a3, v3, amag, work
    full = dict(V=V, rho=rho, nbr_count=cnt, A=A, B=B, gradA=gA, gradB=gB, ax=ax, ay=ay, az=az, dudt=du, pair_count=pc, gradv=gv)
    if full_counts:
        _full_count_check(ps, dict(nbr_count=cnt.cpu().numpy(), pair_count=pc.cpu().numpy()), oracle_mod, label)
    done = 0
    dens, void = int(np.argmin(ps.h)), int(np.argmax(ps.h))
    centres = [(0.5, 0.5, 0.5), (0.0005, 0.9995, 0.5), (float(ps.x[dens]), float(ps.y[dens]), float(ps.z[dens])),
               (float(ps.x[void]), float(ps.y[void]), float(ps.z[void]))]
    for c in centres:
        idx0, _ = wl.select_window(ps, c, 0.01, 0.0)
        if len(idx0) == 0:
            continue
        win = _pick_window(ps, c, 2.5 * float(np.median(ps.h[idx0])))
        if win is None:
            print(f"[parity] {label} window@{np.round(c, 4)} skipped (too many particles in the padded window)")
            continue
        idxp, corep = win
        sub = ps.subset(idxp)
        o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
        od = o.step_derivs(sub)
        sel = torch.from_numpy(idxp).to(dev)
        gs = {k: (v[sel] if v.ndim == 1 else v[:, sel]).cpu().numpy() for k, v in full.items()}
        e_a, e_u = check_parity(sub, gs, od, oracle_gv=o.gradv(), mask=corep, label=f"{label} window@{np.round(c, 4)}")
        print(f"[parity] {label} window n={len(idxp)} core={int(corep.sum())} (h in core {ps.h[idxp][corep].min():.2e}..{ps.h[idxp][corep].max():.2e}): "
              f"dv/dt {e_a:.2e} du/dt {e_u:.2e} momentum {mom:.2e} energy {en:.2e}")
        done += 1
    assert done >= 1


def test_parity_config5_cosmo_large_full(oracle_mod):
    """BASELINE configs[4], zero-indexed reading of "generated as in config 3": the Zel'dovich generator on 512^3 = 134 M
    particles with rms displacement 1.5 spacings.  Its h range is only 1.7x (the k^-2 spectrum puts most of the displacement
    into bulk flows), so it is the large NEAR-LATTICE case; every particle's counts are compared bit-exactly."""
    _large_config_check(wl.make_config("cosmo_large"), oracle_mod, "cosmo512", full_counts=True)


def test_parity_config5_clustered_large(oracle_mod):
    """BASELINE configs[4] read literally ("generated as in config 3 ... strong clustering, h ranging ~20x"): config 3's
    Plummer generator at 512^3 = 134 M particles (32768 spheres), k-th-neighbour h with a range of ~50x.  Windows around the
    densest core, the emptiest void, the box centre and a box corner against the brute-force oracle, invariants on the
    full output.  (No all-particle count check: the oracle's uniform grid is quadratic in the densest cell of a clustered
    set.)  Runs by default (about five and a half minutes, most of it the generator's k-d-tree pass over 134 M points on the
    host); CRK_TEST_LARGE=0 leaves it out, and it is skipped where the host or the GPU is too small to hold the configuration.
    The output of the round-2 run is kept in profiles/r02_config5_clustered_large.md."""
    import os
    if os.environ.get("CRK_TEST_LARGE", "1") == "0":
        pytest.skip("CRK_TEST_LARGE=0: the 134 M-particle clustered configuration was left out on request")
    torch = _torch()
    import psutil
    if psutil.virtual_memory().available < 60e9 or torch.cuda.get_device_properties(0).total_memory < 150e9:
        pytest.skip("the 134 M-particle clustered configuration needs ~60 GB of host memory and ~100 GB on the GPU")
    _large_config_check(wl.make_config("clustered_large"), oracle_mod, "clustered512", full_counts=False)


# ------------------------------------------------------------------------------- NEXT row 1: compatible energy update
@pytest.mark.parametrize("name,n_side,dt", [("tiny_uniform", 16, 1e-3), ("blast_wave", 24, 1e-5), ("clustered", 24, 1e-3),
                                            ("cosmo", 32, 1e-2)])
def test_compatible_energy_parity(name, n_side, dt, oracle_mod):
    """Eqs. 19-23: GPU sweep vs the FP64 oracle, and the exactness property of PAPER.md:141
    (thermal gain = kinetic loss of v -> v + a dt) on the GPU's own accelerations."""
    torch = _torch()
    ps = wl.make_config(name, n_side)
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
    o.step_derivs(ps)
    du_o = o.compatible_energy(dt)
    g = gpu_eval(ps)
    du_g = g["ctx"].compatible_energy(dt)
    torch.cuda.synchronize()
    du_g = du_g.cpu().numpy().astype(np.float64)
    e = rel_l2(du_g, du_o)
    assert e < TOL_DERIV, f"{name} compatible Delta u rel L2 {e:.3e}"
    m = ps.m.astype(np.float64)
    v = np.stack([ps.vx, ps.vy, ps.vz]).astype(np.float64)
    a = np.stack([g["ax"], g["ay"], g["az"]]).astype(np.float64)
    dke = 0.5 * (m * (((v + a * dt) ** 2).sum(0) - (v ** 2).sum(0))).sum()
    res = abs(dke + (m * du_g).sum()) / ((m * np.abs(du_g)).sum() + 1e-300)
    assert res < TOL_INV, f"{name} compatible energy residual {res:.3e}"
    print(f"[parity] {name} n={ps.n} dt={dt}: compatible Delta u {e:.2e}, energy residual {res:.2e}")


def test_compatible_energy_needs_hydro_first():
    torch = _torch()
    from paper_2202_02840_b200 import Crk, CrkError
    ps = wl.tiny_uniform(n_side=8)
    dev = torch.device("cuda:0")
    t = [torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in ("x", "y", "z", "h")]
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h)
    ctx.build_cells(*t)
    with pytest.raises(CrkError):
        ctx.compatible_energy(1e-3)


# ------------------------------------------------------------------------------- NEXT row 3: evolved smoothing length
@pytest.mark.parametrize("name,n_side", [("tiny_uniform", 16), ("clustered", 24), ("cosmo", 32)])
def test_evolved_h_parity(name, n_side, oracle_mod):
    """Eqs. 51-53: the stream pass vs the FP64 oracle; h perturbed so that Delta_N covers both branches"""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    ps = wl.make_config(name, n_side)
    ps.h[:] = (ps.h * np.where(np.arange(ps.n) % 3 == 0, 1.25, np.where(np.arange(ps.n) % 3 == 1, 0.8, 1.0))).astype(np.float32)
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
    o.build(ps.x, ps.y, ps.z, ps.h)
    o.volumes(ps.m)
    h_o = o.evolve_h()
    dev = torch.device("cuda:0")
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in ("x", "y", "z", "h", "m")}
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h)
    ctx.build_cells(t["x"], t["y"], t["z"], t["h"])
    ctx.volumes(t["m"])
    h_g = ctx.evolve_h()
    torch.cuda.synchronize()
    h_g = h_g.cpu().numpy().astype(np.float64)
    e = np.max(np.abs(h_g / h_o - 1))
    assert e < TOL_SCALAR, f"{name} evolved h max rel err {e:.3e}"
    assert (h_o > ps.h).any() and (h_o < ps.h).any()
    print(f"[parity] {name} n={ps.n}: evolved h max rel err {e:.2e}")


# ------------------------------------------------------------------------------- NEXT row 2a: time-step criteria
@pytest.mark.parametrize("name,n_side", [("tiny_uniform", 16), ("blast_wave", 24), ("clustered", 24), ("cosmo", 32)])
def test_timestep_parity(name, n_side, oracle_mod):
    """Eqs. 46-50: maxima reduced inside the momentum sweep + the stream pass, vs the FP64 oracle"""
    torch = _torch()
    from paper_2202_02840_b200 import Crk, CrkError
    ps = wl.make_config(name, n_side)
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
    od = o.step_derivs(ps)
    dt_o, _, _ = o.timestep(0.25)
    dev = torch.device("cuda:0")
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in
         ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")}
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h, timestep=True)
    ctx.build_cells(t["x"], t["y"], t["z"], t["h"])
    ctx.volumes(t["m"])
    ctx.rk_coefficients(want=False)
    ax, ay, az, du, pc = ctx.hydro_derivs(t["vx"], t["vy"], t["vz"], t["u"])
    dt_g = ctx.timestep(0.25)
    torch.cuda.synchronize()
    # the TS variant of the sweep must give the same derivatives
    e_a = rel_l2(np.stack([q.cpu().numpy() for q in (ax, ay, az)]), np.stack([od["ax"], od["ay"], od["az"]]))
    assert e_a < TOL_DERIV
    dt_g = dt_g.cpu().numpy().astype(np.float64)
    fin = np.isfinite(dt_o)
    assert np.array_equal(np.isfinite(dt_g), fin)
    e = np.max(np.abs(dt_g[fin] / dt_o[fin] - 1))
    assert e < TOL_DERIV, f"{name} dt_min max rel err {e:.3e}"
    print(f"[parity] {name} n={ps.n}: dt_min max rel err {e:.2e}, global min {dt_g[fin].min():.3e} (oracle {dt_o[fin].min():.3e})")
    plain = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h)
    plain.build_cells(t["x"], t["y"], t["z"], t["h"])
    with pytest.raises(CrkError):
        plain.timestep(0.25)


# ------------------------------------------------------------------------------- NEXT row 2b: velocity-Verlet step
@pytest.mark.parametrize("name,n_side,dt,steps", [("tiny_uniform", 16, 4e-3, 3), ("clustered", 20, 2e-5, 2), ("cosmo", 32, 2e-3, 2)])
def test_kdk_step_parity(name, n_side, dt, steps, oracle_mod):
    """Eq. 43: crk_kdk_step advances the FP32 state in place; compared with the oracle's FP64 KDK"""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    ps = wl.make_config(name, n_side)
    ref = oracle_mod.kdk_steps(ps, steps, dt)
    dev = torch.device("cuda:0")
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in
         ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")}
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h)
    t2 = {k: v.clone() for k, v in t.items()}
    for _ in range(steps):
        ctx.kdk_step(*[t[k] for k in ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")], dt)
    # CRK_FLAG_KDK_REUSE: follow-up steps reuse the build of the previous step's second evaluation: same bits
    ctx2 = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h, kdk_reuse=True)
    for _ in range(steps):
        ctx2.kdk_step(*[t2[k] for k in ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")], dt)
    torch.cuda.synchronize()
    for k in ("x", "y", "z", "vx", "vy", "vz", "u"):
        assert torch.equal(t[k], t2[k]), f"{name} reuse changed {k}"
    g = {k: v.cpu().numpy().astype(np.float64) for k, v in t.items()}
    for k in ("x", "y", "z"):
        d = np.abs(g[k] - ref[k])
        d = np.minimum(d, ps.box - d)
        assert d.max() < 5e-7 * ps.box, f"{name} {k} max abs err {d.max():.2e}"
        assert (g[k] >= 0).all() and (g[k] < ps.box).all()
    moved = max(np.abs(ref[k] - getattr(ps, k)).max() for k in ("x", "y", "z"))
    e_v = rel_l2(np.stack([g["vx"], g["vy"], g["vz"]]), np.stack([ref["vx"], ref["vy"], ref["vz"]]))
    e_u = rel_l2(g["u"], ref["u"])
    assert e_v < TOL_DERIV and e_u < TOL_DERIV, (e_v, e_u)
    # the step changed something: the velocity change itself must match to 1e-3 of its own size
    dv_g = np.stack([g[q] - getattr(ps, q) for q in ("vx", "vy", "vz")])
    dv_o = np.stack([ref[q] - getattr(ps, q) for q in ("vx", "vy", "vz")])
    e_dv = rel_l2(dv_g, dv_o)
    assert e_dv < 1e-3, e_dv
    assert np.array_equal(g["h"], ps.h) and np.array_equal(g["m"], ps.m)
    print(f"[parity] {name} n={ps.n} {steps} KDK steps dt={dt}: v {e_v:.2e} u {e_u:.2e} dv {e_dv:.2e}, max displacement {moved:.2e}")


# ------------------------------------------------------------------------------- NEXT row 4: paper-default resolution n_h = 4
@pytest.mark.parametrize("name,n_side,grid", [("tiny_uniform", 16, False), ("cosmo", 24, False), ("cosmo", 64, True), ("cosmo", 128, True)])
def test_parity_paper_default_resolution_nh4(name, n_side, grid, oracle_mod):
    """n_h = 4 (N_res = 268 neighbours): every leaf needs a chain of neighbour-list segments (~900
    candidates against 352 slots), which exercises the multi-segment path of the builder and of all sweeps.  The two larger
    cases (262 144 and 2 097 152 particles) compare EVERY particle -- counts bit for bit, all coefficients and derivatives --
    with the oracle run through its grid neighbour search (bit-identical to the brute-force build, tests/test_oracle_pins.py)."""
    ps = wl.make_config(name, n_side)
    ps.h[:] = (ps.h * (4.0 / ps.n_h)).astype(np.float32)
    ps.n_h = 4.0
    assert float(ps.h.max()) < 0.5 * ps.box
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
    od = o.step_derivs(ps, grid=grid)
    g = gpu_eval(ps)
    e_a, e_u = check_parity(ps, g, od, oracle_gv=o.gradv(), label=name + " n_h=4")
    mom, en = check_invariants(ps, g, label=name + " n_h=4")
    seg = g["ctx"].leaf_segments().cpu().numpy()
    multi = float((seg[:, 0] != 0).mean())
    assert multi > 0.9
    print(f"[parity] {name} n_h=4 n={ps.n}: mean neighbours {od['nbr_count'].mean():.0f}, multi-segment leaves {multi:.2f}, "
          f"dv/dt {e_a:.2e} du/dt {e_u:.2e} momentum {mom:.2e} energy {en:.2e}")


def test_parity_non_default_parameters(oracle_mod):
    """box != 1, gamma = 1.4, unequal masses (reading S2), other viscosity constants and n_h: every runtime parameter of
    crk_params reaches the kernels"""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    ps = wl.clustered_plummer(n_side=20)
    L = 2.5
    rng = np.random.default_rng(11)
    for k in ("x", "y", "z", "h"):
        setattr(ps, k, (getattr(ps, k).astype(np.float64) * L).astype(np.float32))
    for k in ("x", "y", "z"):
        a = getattr(ps, k)
        a[a >= np.float32(L)] = np.float32(0.0)
    ps.m = (ps.m * rng.uniform(0.7, 1.3, ps.n)).astype(np.float32)
    ps.box, ps.gamma, ps.n_h = L, 1.4, 3.0       # n_h enters through hhat, eta_crit, eta_fold only: the 58 neighbours stay
    kw = dict(C_l=1.0, C_q=2.5, eps=0.05)
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h, **kw)
    od = o.step_derivs(ps)
    dev = torch.device("cuda:0")
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in
         ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")}
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h, timestep=True, **kw)
    ctx.build_cells(t["x"], t["y"], t["z"], t["h"])
    V, rho, cnt = ctx.volumes(t["m"])
    A, B, gA, gB = ctx.rk_coefficients()
    ax, ay, az, du, pc = ctx.hydro_derivs(t["vx"], t["vy"], t["vz"], t["u"])
    g = dict(V=V, rho=rho, nbr_count=cnt, A=A, B=B, gradA=gA, gradB=gB, ax=ax, ay=ay, az=az, dudt=du, pair_count=pc,
             gradv=ctx.gradv())
    dt_g = ctx.timestep(0.3)
    du_c = ctx.compatible_energy(1e-4)
    torch.cuda.synchronize()
    g = {k: v.cpu().numpy() for k, v in g.items()}
    e_a, e_u = check_parity(ps, g, od, oracle_gv=o.gradv(), label="non-default params")
    mom, en = check_invariants(ps, g, label="non-default params")
    dt_o, _, _ = o.timestep(0.3)
    fin = np.isfinite(dt_o)
    assert np.max(np.abs(dt_g.cpu().numpy()[fin] / dt_o[fin] - 1)) < TOL_DERIV
    assert rel_l2(du_c.cpu().numpy().astype(np.float64), o.compatible_energy(1e-4)) < TOL_DERIV
    print(f"[parity] non-default params n={ps.n}: dv/dt {e_a:.2e} du/dt {e_u:.2e} momentum {mom:.2e} energy {en:.2e}")


def test_parity_config4_cosmo_every_particle(oracle_mod):
    """BASELINE configs[3] (256^3, the bench workload): EVERY particle against the FP64 oracle run on the full
    configuration through its grid neighbour search (bit-identical to the brute-force oracle, tests/test_oracle_pins.py)"""
    ps = wl.make_config("cosmo")
    o = oracle_mod.Oracle(ps.box, ps.gamma, ps.n_h)
    od = o.step_derivs(ps, grid=True)
    g = gpu_eval(ps)
    e_a, e_u = check_parity(ps, g, od, oracle_gv=o.gradv(), label="cosmo256 all particles")
    mom, en = check_invariants(ps, g, label="cosmo256 all particles")
    a_o = np.stack([od["ax"], od["ay"], od["az"]]); a_g = np.stack([g["ax"], g["ay"], g["az"]]).astype(np.float64)
    worst = np.sqrt(((a_g - a_o) ** 2).sum(0)).max() / np.sqrt((a_o ** 2).sum(0).mean())
    print(f"[parity] cosmo256 all {ps.n} particles: dv/dt {e_a:.2e} du/dt {e_u:.2e} (worst particle {worst:.2e} of rms) "
          f"momentum {mom:.2e} energy {en:.2e}")
    assert worst < 1e-3


# ------------------------------------------------------------------------------- integration: Sod shock tube
def _sod_exact(x_over_t, gamma, rl, pl, rr, pr):
    """exact solution of the Riemann problem for an ideal gas at rest on both sides (textbook two-shock/rarefaction
    iteration; left state high pressure): density, velocity, pressure at the similarity coordinate x/t"""
    g = gamma
    cl, cr = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)

    def f(p, rk, pk, ck):
        if p > pk:      # shock
            A, B = 2.0 / ((g + 1) * rk), (g - 1) / (g + 1) * pk
            return (p - pk) * np.sqrt(A / (p + B))
        return 2 * ck / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1)      # rarefaction

    lo, hi = 1e-8, max(pl, pr)
    for _ in range(200):
        p = 0.5 * (lo + hi)
        if f(p, rl, pl, cl) + f(p, rr, pr, cr) > 0:
            hi = p
        else:
            lo = p
    ps = 0.5 * (lo + hi)
    us = 0.5 * (f(ps, rr, pr, cr) - f(ps, rl, pl, cl))
    rsl = rl * (ps / pl) ** (1 / g)                                              # behind the left rarefaction
    csl = cl * (ps / pl) ** ((g - 1) / (2 * g))
    rsr = rr * ((ps / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pr + 1))   # behind the right shock
    S = cr * np.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))            # shock speed
    s = np.asarray(x_over_t, dtype=np.float64)
    rho = np.where(s < -cl, rl, np.where(s < us - csl, 0.0, np.where(s < us, rsl, np.where(s < S, rsr, rr))))
    fan = (s >= -cl) & (s < us - csl)
    cfan = 2 / (g + 1) * (cl - (g - 1) / 2 * s)
    rho = np.where(fan, rl * (cfan / cl) ** (2 / (g - 1)), rho)
    u = np.where(s < -cl, 0.0, np.where(fan, 2 / (g + 1) * (cl + s), np.where(s < S, us, 0.0)))
    return rho, u, S, us


@pytest.mark.parametrize("compatible", [False, True])
def test_sod_shock_tube_with_kdk_timestep_and_evolved_h(compatible):
    """The next rows working together (Eq. 43 steps, Eqs. 46-50 time steps, Eqs. 51-53 smoothing lengths) on the paper's Sod
    set-up (rho_h = P_h = 1, rho_l = P_l = 1/8, gamma = 5/3, two interfaces in a periodic domain, step
    function IC, here at half scale: unit box, interfaces at 0.25 / 0.75, t = 0.075), against the exact Riemann solution.
    A physics check, not a parity check: tolerances are those of a 96-cell first-order shock capture."""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    ns, gamma, n_h = 96, 5.0 / 3.0, 2.4
    q = (np.arange(ns) + 0.5) / ns
    X = np.stack(np.meshgrid(q, q, q, indexing="ij")).reshape(3, -1)
    n = X.shape[1]
    high = (X[0] >= 0.25) & (X[0] < 0.75)
    rho0 = np.where(high, 1.0, 0.125)
    P0 = np.where(high, 1.0, 0.125)
    dev = torch.device("cuda:0")
    f32 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
    x, y, z = f32(X[0]), f32(X[1]), f32(X[2])
    m = f32(rho0 / ns ** 3)
    u = f32(P0 / ((gamma - 1) * rho0))
    vx, vy, vz = (torch.zeros(n, device=dev) for _ in range(3))
    h = torch.full((n,), n_h / ns, device=dev)
    ctx = Crk(box=1.0, gamma=gamma, n_h=n_h, timestep=True, kdk_compatible=compatible)
    ctx.step_derivs(x, y, z, h, vx, vy, vz, m, u)
    t, t_end, steps = 0.0, 0.075, 0
    e0 = float((m.double() * (u.double() + 0.5 * (vx.double() ** 2 + vy.double() ** 2 + vz.double() ** 2))).sum())
    while t < t_end - 1e-12:
        dt = min(float(ctx.timestep(0.25).min()), t_end - t)
        ctx.kdk_step(x, y, z, h, vx, vy, vz, m, u, dt)
        h.copy_(ctx.evolve_h())                      # volumes of the new positions are resident after the step
        t += dt
        steps += 1
        assert steps < 2000
    ctx.build_cells(x, y, z, h)
    V, rho, cnt = ctx.volumes(m)
    torch.cuda.synchronize()
    e1 = float((m.double() * (u.double() + 0.5 * (vx.double() ** 2 + vy.double() ** 2 + vz.double() ** 2))).sum())
    xs, rs, us_ = x.cpu().numpy().astype(np.float64), rho.cpu().numpy().astype(np.float64), vx.cpu().numpy().astype(np.float64)
    sel = (xs >= 0.52) & (xs < 0.98)                 # the right-moving tube around the interface at 0.75
    re, ue, S, ustar = _sod_exact((xs[sel] - 0.75) / t_end, gamma, 1.0, 1.0, 0.125, 0.125)
    l1_rho = np.abs(rs[sel] - re).mean() / re.mean()
    l1_u = np.abs(us_[sel] - ue).mean() / ustar
    # planar symmetry: the compressed cubic lattice re-arranges behind the shock (round-off seeded), but the transverse
    # motion stays a small fraction of the flow speed
    vt = float(torch.sqrt((vy.double() ** 2 + vz.double() ** 2).mean()))
    nb = float(cnt.float().mean())
    print(f"[sod] compatible={compatible} n={n} steps={steps}: L1(rho) {l1_rho:.3f} L1(u)/u* {l1_u:.3f}, shock speed {S:.3f}, u* {ustar:.3f}, "
          f"rms transverse speed {vt:.1e}, energy drift {abs(e1 / e0 - 1):.1e}, mean neighbours {nb:.1f}")
    assert l1_rho < 0.08 and l1_u < 0.15
    assert vt < 0.05 * ustar
    assert abs(e1 / e0 - 1) < (2e-6 if compatible else 2e-3)     # Eqs. 19-23 conserve to roundoff, Eq. 18 to O(dt^2)
    assert 50 < nb < 66


@pytest.mark.parametrize("name,n_side,dt,steps", [("tiny_uniform", 16, 4e-3, 3), ("cosmo", 32, 2e-3, 2)])
def test_kdk_step_with_compatible_energy(name, n_side, dt, steps, oracle_mod):
    """CRK_FLAG_KDK_COMPATIBLE (reading S20): Verlet step whose half kicks use Eqs. 19-23; against the oracle's FP64
    version, and total energy conserved to FP32 roundoff on the GPU"""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    ps = wl.make_config(name, n_side)
    ref = oracle_mod.kdk_steps(ps, steps, dt, compatible=True)
    dev = torch.device("cuda:0")
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in
         ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")}
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h, kdk_compatible=True, kdk_reuse=True)
    m = t["m"].double()
    energy = lambda: float((m * (t["u"].double() + 0.5 * (t["vx"].double() ** 2 + t["vy"].double() ** 2 + t["vz"].double() ** 2))).sum())
    e0 = energy()
    for _ in range(steps):
        ctx.kdk_step(*[t[k] for k in ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")], dt)
    torch.cuda.synchronize()
    e1 = energy()
    g = {k: v.cpu().numpy().astype(np.float64) for k, v in t.items()}
    e_v = rel_l2(np.stack([g["vx"], g["vy"], g["vz"]]), np.stack([ref["vx"], ref["vy"], ref["vz"]]))
    e_u = rel_l2(g["u"], ref["u"])
    du_g, du_o = g["u"] - ps.u, ref["u"] - ps.u
    e_du = rel_l2(du_g, du_o)
    assert e_v < TOL_DERIV and e_u < TOL_DERIV and e_du < 1e-3, (e_v, e_u, e_du)
    drift = abs(e1 / e0 - 1)
    assert drift < 2e-6, drift
    print(f"[parity] {name} n={ps.n} {steps} compatible KDK steps: v {e_v:.2e} u {e_u:.2e} du {e_du:.2e}, energy drift {drift:.1e}")


def test_sedov_blast_wave_shock_radius():
    """BASELINE config 2 evolved for real: 64^3 blast wave with the Verlet step, the compatible energy,
    the time-step criteria and the evolved smoothing length; the shock radius follows the Sedov-Taylor similarity
    solution R = xi0 (E t^2 / rho)^(1/5), xi0 = 1.152 for gamma = 5/3.  A physics check."""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    ps = wl.make_config("blast_wave")
    dev = torch.device("cuda:0")
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in
         ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")}
    arg = lambda: [t[k] for k in ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")]
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h, timestep=True, kdk_compatible=True)
    ctx.step_derivs(*arg())
    m = t["m"].double()
    energy = lambda: float((m * (t["u"].double() + 0.5 * (t["vx"].double() ** 2 + t["vy"].double() ** 2 + t["vz"].double() ** 2))).sum())
    e0 = energy()
    time, t_end, steps = 0.0, 0.04, 0
    while time < t_end - 1e-12:
        dt = min(float(ctx.timestep(0.25).min()), t_end - time)
        ctx.kdk_step(*arg(), dt)
        t["h"].copy_(ctx.evolve_h())
        time += dt
        steps += 1
        assert steps < 5000
    ctx.build_cells(t["x"], t["y"], t["z"], t["h"])
    V, rho, cnt = ctx.volumes(t["m"])
    torch.cuda.synchronize()
    e1 = energy()
    X = np.stack([t[k].cpu().numpy().astype(np.float64) for k in ("x", "y", "z")]) - 0.5
    r = np.sqrt((X ** 2).sum(0))
    rh = rho.cpu().numpy().astype(np.float64)
    bins = np.linspace(0.05, 0.48, 44)
    idx = np.digitize(r, bins)
    prof = np.array([np.median(rh[idx == b]) if (idx == b).sum() > 20 else 0.0 for b in range(1, len(bins))])
    r_peak = 0.5 * (bins[:-1] + bins[1:])[np.argmax(prof)]
    r_exact = 1.152 * (1.0 * t_end ** 2 / 1.0) ** 0.2
    umin = float(t["u"].min())
    print(f"[sedov] steps={steps} shock radius {r_peak:.3f} (similarity solution {r_exact:.3f}), peak density {prof.max():.2f}, "
          f"energy drift {abs(e1 / e0 - 1):.1e}, min u {umin:.2e}")
    assert abs(r_peak / r_exact - 1) < 0.06
    assert 1.8 < prof.max() < 4.0            # strong-shock limit (gamma + 1)/(gamma - 1) = 4, smeared at this resolution
    assert abs(e1 / e0 - 1) < 1e-5


def test_results_are_bit_reproducible():
    """no atomics in any sum, fixed-order reductions: two evaluations (fresh contexts) give identical bits"""
    torch = _torch()
    from paper_2202_02840_b200 import Crk
    ps = wl.make_config("clustered", 24)
    dev = torch.device("cuda:0")
    t = [torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")]
    runs = []
    for _ in range(2):
        ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h, timestep=True)
        out = ctx.step_derivs(*t)
        runs.append([o.clone() for o in out] + [ctx.compatible_energy(1e-3).clone(), ctx.timestep(0.25).clone()])
    torch.cuda.synchronize()
    for a, b in zip(*runs):
        assert torch.equal(a, b)
