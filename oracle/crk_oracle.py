"""ctypes front end of the CPU oracle (oracle/crk_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)
sys.path.pop(0)


class _Params(C.Structure):
    _fields_ = [("box", C.c_double), ("gamma", C.c_double), ("n_h", C.c_double),
                ("C_l", C.c_double), ("C_q", C.c_double), ("eps", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        fp, dp, up = C.POINTER(C.c_float), C.POINTER(C.c_double), C.POINTER(C.c_uint32)
        L.crk_oracle_create.restype = C.c_void_p
        L.crk_oracle_create.argtypes = [C.POINTER(_Params)]
        L.crk_oracle_destroy.argtypes = [C.c_void_p]
        L.crk_oracle_set_threads.argtypes = [C.c_int]
        L.crk_oracle_get_threads.restype = C.c_int
        L.crk_oracle_build.argtypes = [C.c_void_p, C.c_int64, fp, fp, fp, fp]
        L.crk_oracle_build_grid.argtypes = [C.c_void_p, C.c_int64, fp, fp, fp, fp]
        L.crk_oracle_volumes.argtypes = [C.c_void_p, fp, dp, dp, up]
        L.crk_oracle_rk_coefficients.argtypes = [C.c_void_p, dp, dp, dp, dp]
        L.crk_oracle_hydro_derivs.argtypes = [C.c_void_p, fp, fp, fp, fp, dp, dp, dp, dp, up]
        L.crk_oracle_hydro_derivs_active.argtypes = [C.c_void_p, C.POINTER(C.c_uint8), fp, fp, fp, fp, dp, dp, dp, dp]
        L.crk_oracle_W.restype = C.c_double
        L.crk_oracle_W.argtypes = [C.c_double, C.c_double]
        L.crk_oracle_dWdr.restype = C.c_double
        L.crk_oracle_dWdr.argtypes = [C.c_double, C.c_double]
        L.crk_oracle_get_moments.argtypes = [C.c_void_p, dp, dp, dp]
        L.crk_oracle_get_gradv.argtypes = [C.c_void_p, dp]
        L.crk_oracle_rk_sums.argtypes = [C.c_void_p, dp, dp, dp, dp]
        L.crk_oracle_eval_AB_at.argtypes = [C.c_void_p, dp, C.c_double, dp, dp]
        L.crk_oracle_pair_term.argtypes = [C.c_void_p, C.c_int64, C.c_int64, dp]
        L.crk_oracle_pair_visc.argtypes = [C.c_void_p, C.c_int64, C.c_int64, dp]
        L.crk_oracle_compatible_energy.argtypes = [C.c_void_p, C.c_double, dp]
        L.crk_oracle_compatible_energy_kick.argtypes = [C.c_void_p, C.c_double, dp, dp]
        L.crk_oracle_evolve_h.argtypes = [C.c_void_p, dp]
        L.crk_oracle_grid_counts.argtypes = [C.c_double, C.c_int64, fp, fp, fp, fp, up, up]
        L.crk_oracle_timestep.argtypes = [C.c_void_p, C.c_double, dp, dp, dp]
        L.crk_oracle_h_update.argtypes = [C.c_double, C.c_double, C.c_double]
        L.crk_oracle_h_update.restype = C.c_double
        L.crk_oracle_pair_compat.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_double, dp]
        L.crk_oracle_neighbors.restype = C.c_int64
        L.crk_oracle_neighbors.argtypes = [C.c_void_p, C.c_int64, up, C.c_int64]
        _lib = L
    return _lib


def _f(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(C.POINTER(C.c_float))


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _u(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint32))


def kernel_W(r, h):
    return lib().crk_oracle_W(float(r), float(h))


def kernel_dWdr(r, h):
    return lib().crk_oracle_dWdr(float(r), float(h))


def set_threads(n: int):
    lib().crk_oracle_set_threads(int(n))


def get_threads() -> int:
    return int(lib().crk_oracle_get_threads())


class Oracle:
    """Call-by-call mirror of the C-ABI library: build -> volumes -> rk_coefficients -> hydro_derivs."""

    def __init__(self, box=1.0, gamma=5.0 / 3.0, n_h=2.4, C_l=2.0, C_q=1.0, eps=0.1):
        self.params = _Params(box, gamma, n_h, C_l, C_q, eps)
        self._c = lib().crk_oracle_create(C.byref(self.params))
        self.n = 0
        self._keep = []

    def __del__(self):
        if getattr(self, "_c", None):
            lib().crk_oracle_destroy(self._c)
            self._c = None

    def build(self, x, y, z, h, grid=False):
        """grid=True: same neighbour structure through the uniform grid (oracle at scale) instead of the O(N^2) scan"""
        (x, px), (y, py), (z, pz), (h, ph) = _f(x), _f(y), _f(z), _f(h)
        self.n = x.shape[0]
        rc = (lib().crk_oracle_build_grid if grid else lib().crk_oracle_build)(self._c, self.n, px, py, pz, ph)
        if rc == -2:
            raise RuntimeError("crk_oracle_build_grid: fewer than 3 cells per side (use the brute-force build)")
        if rc:
            raise ValueError("crk_oracle_build: bad input (h<=0, h>=L/2 or position outside [0,L))")

    def volumes(self, m):
        m, pm = _f(m)
        n = self.n
        V, rho, cnt = np.empty(n), np.empty(n), np.empty(n, dtype=np.uint32)
        rc = lib().crk_oracle_volumes(self._c, pm, _d(V), _d(rho), _u(cnt))
        assert rc == 0
        return V, rho, cnt

    def rk_coefficients(self):
        n = self.n
        A, B, gA, gB = np.empty(n), np.empty((3, n)), np.empty((3, n)), np.empty((9, n))
        rc = lib().crk_oracle_rk_coefficients(self._c, _d(A), _d(B), _d(gA), _d(gB))
        assert rc == 0
        return A, B, gA, gB

    def hydro_derivs(self, vx, vy, vz, u):
        (vx, p1), (vy, p2), (vz, p3), (u, p4) = _f(vx), _f(vy), _f(vz), _f(u)
        n = self.n
        ax, ay, az, du = np.empty(n), np.empty(n), np.empty(n), np.empty(n)
        cnt = np.empty(n, dtype=np.uint32)
        rc = lib().crk_oracle_hydro_derivs(self._c, p1, p2, p3, p4, _d(ax), _d(ay), _d(az), _d(du), _u(cnt))
        assert rc == 0
        return ax, ay, az, du, cnt

    def hydro_derivs_active(self, active, vx, vy, vz, u):
        """Eqs. 17-18 for the particles with active[i] != 0 only (NaN elsewhere)"""
        (vx, p1), (vy, p2), (vz, p3), (u, p4) = _f(vx), _f(vy), _f(vz), _f(u)
        act = np.ascontiguousarray(active, dtype=np.uint8)
        n = self.n
        ax, ay, az, du = np.empty(n), np.empty(n), np.empty(n), np.empty(n)
        rc = lib().crk_oracle_hydro_derivs_active(self._c, act.ctypes.data_as(C.POINTER(C.c_uint8)), p1, p2, p3, p4,
                                                  _d(ax), _d(ay), _d(az), _d(du))
        assert rc == 0
        return ax, ay, az, du

    def step_derivs(self, ps, grid=False):
        """ps: crk_workloads.ParticleSet (or anything with x,y,z,h,vx,vy,vz,m,u). Returns dict of all outputs."""
        self.build(ps.x, ps.y, ps.z, ps.h, grid=grid)
        V, rho, nbr = self.volumes(ps.m)
        A, B, gA, gB = self.rk_coefficients()
        ax, ay, az, du, pc = self.hydro_derivs(ps.vx, ps.vy, ps.vz, ps.u)
        return dict(V=V, rho=rho, nbr_count=nbr, A=A, B=B, gradA=gA, gradB=gB,
                    ax=ax, ay=ay, az=az, dudt=du, pair_count=pc)

    def timestep(self, C_cfl=0.25):
        """Eqs. 46-50 after hydro_derivs: (dt_min, dt_hyd, dt_acc) per particle"""
        a, b, c = np.empty(self.n), np.empty(self.n), np.empty(self.n)
        assert lib().crk_oracle_timestep(self._c, float(C_cfl), _d(a), _d(b), _d(c)) == 0
        return a, b, c

    def evolve_h(self):
        """Eqs. 51-53 after volumes(): the adjusted support radii"""
        h = np.empty(self.n)
        assert lib().crk_oracle_evolve_h(self._c, _d(h)) == 0
        return h

    def compatible_energy(self, dt):
        """Eqs. 19-23: Delta u over dt from the pairwise accelerations of the last hydro_derivs"""
        du = np.empty(self.n)
        assert lib().crk_oracle_compatible_energy(self._c, float(dt), _d(du)) == 0
        return du

    def compatible_energy_kick(self, dt, kick):
        """Eqs. 19-21, 23 for a kick with velocity change kick[3][n] = v' - v over dt (v = velocities of the last hydro_derivs)"""
        kick = np.ascontiguousarray(kick, dtype=np.float64)
        assert kick.shape == (3, self.n)
        du = np.empty(self.n)
        assert lib().crk_oracle_compatible_energy_kick(self._c, float(dt), _d(kick), _d(du)) == 0
        return du

    def pair_compat(self, i, j, dt):
        out = np.empty(3)
        assert lib().crk_oracle_pair_compat(self._c, int(i), int(j), float(dt), _d(out)) == 0
        return out   # du_ij, dE_ij, f_ij

    # ---- diagnostics for the pins
    def moments(self):
        n = self.n
        m0, m1, m2 = np.empty(n), np.empty((3, n)), np.empty((9, n))
        assert lib().crk_oracle_get_moments(self._c, _d(m0), _d(m1), _d(m2)) == 0
        return m0, m1, m2

    def gradv(self):
        g = np.empty((9, self.n))
        assert lib().crk_oracle_get_gradv(self._c, _d(g)) == 0
        return g

    def rk_sums(self):
        n = self.n
        S0, S1, G0, G1 = np.empty(n), np.empty((3, n)), np.empty((3, n)), np.empty((9, n))
        assert lib().crk_oracle_rk_sums(self._c, _d(S0), _d(S1), _d(G0), _d(G1)) == 0
        return S0, S1, G0, G1

    def eval_AB_at(self, p, h):
        p = np.ascontiguousarray(p, dtype=np.float64)
        A = C.c_double()
        B = np.empty(3)
        assert lib().crk_oracle_eval_AB_at(self._c, _d(p), float(h), C.byref(A), _d(B)) == 0
        return A.value, B

    def pair_term(self, i, j):
        out = np.empty(4)
        assert lib().crk_oracle_pair_term(self._c, int(i), int(j), _d(out)) == 0
        return out

    def pair_visc(self, i, j):
        out = np.empty(5)
        assert lib().crk_oracle_pair_visc(self._c, int(i), int(j), _d(out)) == 0
        return out

    def neighbors(self, i):
        cnt = lib().crk_oracle_neighbors(self._c, int(i), None, 0)
        buf = np.empty(max(cnt, 1), dtype=np.uint32)
        lib().crk_oracle_neighbors(self._c, int(i), _u(buf), cnt)
        buf = buf[:cnt]
        return buf & np.uint32(0x3fffffff), (buf >> np.uint32(31)).astype(bool), ((buf >> np.uint32(30)) & 1).astype(bool)


def euler_steps(ps, n_steps: int, dt: float, oracle: Oracle | None = None, grid: bool = False):
    """Step 12 of DESIGN.md (BASELINE config 2): forward Euler in FP64 on the oracle's derivatives.
    Yields (step, state_f32 ParticleSet-like dict, derivs dict) BEFORE each update, so a caller can
    teacher-force another implementation on the same FP32 state.  h and m stay fixed.
    grid=True: neighbours through crk_oracle_build_grid (bit-identical structure, pinned) so that 64^3 takes seconds."""
    import copy
    o = oracle or Oracle(ps.box, ps.gamma, ps.n_h)
    st = {k: np.asarray(getattr(ps, k), dtype=np.float64).copy() for k in ("x", "y", "z", "vx", "vy", "vz", "u")}
    L = ps.box
    for step in range(n_steps + 1):
        cur = copy.copy(ps)
        for k in st:
            setattr(cur, k, st[k].astype(np.float32))
        for k in ("x", "y", "z"):           # the float32 cast may round up to L
            a = getattr(cur, k)
            a[a >= np.float32(L)] = np.float32(0.0)
        d = o.step_derivs(cur, grid=grid)
        yield step, cur, d
        if step == n_steps:
            break
        for k, v, a in (("x", "vx", "ax"), ("y", "vy", "ay"), ("z", "vz", "az")):
            p = st[k] + st[v] * dt
            st[k] = p - np.floor(p / L) * L          # re-wrap with floor (reading S12)
            st[v] = st[v] + d[a] * dt
        st["u"] = st["u"] + d["dudt"] * dt


def _f32_state(ps, st, L):
    import copy
    cur = copy.copy(ps)
    for k in st:
        setattr(cur, k, st[k].astype(np.float32))
    for k in ("x", "y", "z"):           # the float32 cast may round up to L
        a = getattr(cur, k)
        a[a >= np.float32(L)] = np.float32(0.0)
    return cur


def kdk_steps(ps, n_steps: int, dt: float, oracle: Oracle | None = None, compatible: bool = False):
    """NEXT row 2b: the hydro-only velocity-Verlet operator U_V of Eq. 43 with a = 1, dt/dy = 1,
    p = v, in FP64 on the oracle's derivatives (each evaluation sees the float32 cast of the state, like the library):
        v^1/2 = v^0 + (1/2) a(x^0, v^0, u^0) dt          u^1/2 = u^0 + (1/2) udot(x^0, v^0, u^0) dt
        x^1   = x^0 + v^1/2 dt  (wrapped into [0, L))
        v_p   = v^1/2 + (1/2) a(x^0, v^0, u^0) dt        u_p   = u^1/2 + (1/2) udot(x^0, v^0, u^0) dt     (predictions)
        v^1   = v^1/2 + (1/2) a(x^1, v_p, u_p) dt        u^1   = u^1/2 + (1/2) udot(x^1, v_p, u_p) dt
    Reading S19: the "Delta u" of Eq. 43 is taken as (du/dt of Eq. 18) dt.  h and m stay fixed.
    compatible=True (reading S20): the two half kicks use the compatible energy of Eqs. 19-23 instead, each for its own
    velocity change: Delta u_1 for v^0 -> v^1/2 with the pair accelerations of the first evaluation, Delta u_2 for
    v^1/2 -> v^1 with those of the second (which was taken at v_p = v^1/2 + a^0 dt/2, so relative to that state the kick
    v^1/2 + v^1 = 2 v_p + (a^1 dt/2 - a^0 dt)); u_p = u^1/2 + Delta u_1.  Total energy is then conserved to roundoff.
    Returns the FP64 state dict after n_steps."""
    o = oracle or Oracle(ps.box, ps.gamma, ps.n_h)
    st = {k: np.asarray(getattr(ps, k), dtype=np.float64).copy() for k in ("x", "y", "z", "vx", "vy", "vz", "u")}
    L = ps.box
    ax = (("x", "vx", "ax"), ("y", "vy", "ay"), ("z", "vz", "az"))
    for _ in range(n_steps):
        d0 = o.step_derivs(_f32_state(ps, st, L))
        half = {v: st[v] + 0.5 * d0[a] * dt for _, v, a in ax}
        if compatible:
            du1 = o.compatible_energy_kick(0.5 * dt, np.stack([0.5 * dt * d0[a] for _, _, a in ax]))
        else:
            du1 = 0.5 * d0["dudt"] * dt
        u_half = st["u"] + du1
        pred = dict(st)
        for k, v, a in ax:
            p = st[k] + half[v] * dt
            pred[k] = p - np.floor(p / L) * L
            pred[v] = half[v] + 0.5 * d0[a] * dt
        pred["u"] = u_half + du1
        d1 = o.step_derivs(_f32_state(ps, pred, L))
        for k, v, a in ax:
            st[k] = pred[k]
            st[v] = half[v] + 0.5 * d1[a] * dt
        if compatible:
            du2 = o.compatible_energy_kick(0.5 * dt, np.stack([0.5 * dt * d1[a] - dt * d0[a] for _, _, a in ax]))
        else:
            du2 = 0.5 * d1["dudt"] * dt
        st["u"] = u_half + du2
    return st


def grid_counts(ps):
    """oracle at scale: (nbr_count, pair_count) of every particle of a full configuration (uniform grid of cells >= h_max,
    same FP32 predicate as the brute-force build)"""
    n = ps.n
    a, b = np.empty(n, dtype=np.uint32), np.empty(n, dtype=np.uint32)
    arrs = [np.ascontiguousarray(getattr(ps, k), dtype=np.float32) for k in ("x", "y", "z", "h")]
    rc = lib().crk_oracle_grid_counts(float(ps.box), n, *[_f(q)[1] for q in arrs], _u(a), _u(b))
    if rc != 0:
        raise RuntimeError(f"crk_oracle_grid_counts failed ({rc})")
    return a, b


def h_update(h, n_i, n_h):
    """Eqs. 51-53 for one particle (number density n_i)"""
    return lib().crk_oracle_h_update(float(h), float(n_i), float(n_h))
