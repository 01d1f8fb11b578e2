"""ctypes loader of the CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, bench.py's cpu_baseline / --impl reference legs and __graft_entry__.smoke() may
import this.  It shares no code with paper_2308_16597_b200.binding.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
if _HERE not in sys.path:
    sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_bp = C.POINTER(C.c_ubyte)


class OracleParams(C.Structure):
    _fields_ = [("nu", C.c_double), ("kappa", C.c_double), ("rho0", C.c_double),
                ("T0", C.c_double), ("g", C.c_double), ("gbeta", C.c_double),
                ("body_ax", C.c_double), ("body_ay", C.c_double), ("periodic_x", C.c_int),
                ("wall_T_type", C.c_int * 4), ("wall_T", C.c_double * 4),
                ("rep_s", C.c_double), ("rep_eps", C.c_double), ("rep_power", C.c_int),
                ("max_particles", C.c_int), ("max_links_per_particle", C.c_int)]

    @classmethod
    def from_dict(cls, d):
        p = cls()
        for k, _ in cls._fields_:
            v = d[k]
            if k == "wall_T_type":
                p.wall_T_type = (C.c_int * 4)(*[int(t) for t in v])
            elif k == "wall_T":
                p.wall_T = (C.c_double * 4)(*[float(t) for t in v])
            else:
                setattr(p, k, v)
        return p


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        L = _lib
        L.oracle_last_error.restype = C.c_char_p
        L.oracle_link_q_ellipse.restype = C.c_double
        L.oracle_link_q_ellipse.argtypes = [C.c_double, C.c_double, C.c_int] + [C.c_double] * 6
        L.oracle_rotate_unit.restype = None
        L.oracle_rotate_unit.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_double]
        L.oracle_link_q.restype = C.c_double
        L.oracle_link_q.argtypes = [C.c_double, C.c_double, C.c_int, C.c_double, C.c_double, C.c_double]
        L.oracle_bounce_back_f.restype = C.c_double
        L.oracle_bounce_back_f.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_double,
                                           C.c_double, C.c_double, C.c_int, C.c_double, C.c_double,
                                           C.c_double]
        L.oracle_bounce_back_g.restype = C.c_double
        L.oracle_bounce_back_g.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_double,
                                           C.c_int, C.c_double, C.c_double]
        L.oracle_repulsion_mag.restype = C.c_double
        L.oracle_repulsion_mag.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, C.c_int]
        L.oracle_refill_direction.restype = C.c_int
        L.oracle_refill_direction.argtypes = [C.c_double, C.c_double]
        L.oracle_feq.argtypes = [C.c_double, C.c_double, C.c_double, _dp]
        L.oracle_geq.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, _dp]
        L.oracle_relaxation_rates.argtypes = [C.c_double, C.c_double, _dp, _dp, _dp]
        L.oracle_integrate.argtypes = [_dp, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double]
        L.oracle_momentum_exchange.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double,
                                               C.c_double, C.c_double, C.c_double, _dp]
        L.oracle_refill_f.argtypes = [C.c_int, _dp, _dp, _dp, C.c_double, C.c_double, C.c_double, _dp]
        L.oracle_ellipse_normal.restype = None
        L.oracle_ellipse_normal.argtypes = [C.c_double] * 6 + [_dp, _dp]
        L.oracle_set_state.argtypes = [C.c_void_p, _dp, _dp, C.c_int] + [_dp] * 6
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _arr(n):
    return np.empty(n, dtype=np.float64)


# ---- pieces -------------------------------------------------------------------------------
def feq(rho, ux, uy):
    o = _arr(9)
    lib().oracle_feq(rho, ux, uy, _d(o))
    return o


def geq(T, ux, uy, kappa):
    o = _arr(5)
    lib().oracle_geq(T, ux, uy, kappa, _d(o))
    return o


def moments_f(f):
    f = np.ascontiguousarray(f, dtype=np.float64)
    o = _arr(9)
    lib().oracle_moments_f(_d(f), _d(o))
    return o


def moments_g(g):
    g = np.ascontiguousarray(g, dtype=np.float64)
    o = _arr(5)
    lib().oracle_moments_g(_d(g), _d(o))
    return o


def from_moments_f(m):
    m = np.ascontiguousarray(m, dtype=np.float64)
    o = _arr(9)
    lib().oracle_from_moments_f(_d(m), _d(o))
    return o


def from_moments_g(m):
    m = np.ascontiguousarray(m, dtype=np.float64)
    o = _arr(5)
    lib().oracle_from_moments_g(_d(m), _d(o))
    return o


def relaxation_rates(nu, kappa):
    S, Q, aT = _arr(9), _arr(5), C.c_double()
    lib().oracle_relaxation_rates(nu, kappa, _d(S), _d(Q), C.byref(aT))
    return S, Q, aT.value


def macroscopic(params, f, g):
    P = OracleParams.from_dict(params)
    f = np.ascontiguousarray(f, dtype=np.float64)
    g = np.ascontiguousarray(g, dtype=np.float64)
    r, ux, uy, T = C.c_double(), C.c_double(), C.c_double(), C.c_double()
    lib().oracle_macroscopic(C.byref(P), _d(f), _d(g), C.byref(r), C.byref(ux), C.byref(uy), C.byref(T))
    return r.value, ux.value, uy.value, T.value


def collide_node(params, f, g):
    P = OracleParams.from_dict(params)
    f = np.ascontiguousarray(f, dtype=np.float64)
    g = np.ascontiguousarray(g, dtype=np.float64)
    fo, go = _arr(9), _arr(5)
    lib().oracle_collide_node(C.byref(P), _d(f), _d(g), _d(fo), _d(go))
    return fo, go


def link_q(xf, yf, alpha, xc, yc, r):
    return lib().oracle_link_q(xf, yf, alpha, xc, yc, r)


def link_q_ellipse(xf, yf, alpha, xc, yc, a, b, c, s):
    return lib().oracle_link_q_ellipse(xf, yf, alpha, xc, yc, a, b, c, s)


def rotate_unit(c, s, d):
    cc, ss = C.c_double(c), C.c_double(s)
    lib().oracle_rotate_unit(C.byref(cc), C.byref(ss), d)
    return cc.value, ss.value


def bounce_back_f(alpha, q, fi_0, fi_1, fi_2, fib_0, fib_1, nbehind, rho0, uwx, uwy):
    return lib().oracle_bounce_back_f(alpha, q, fi_0, fi_1, fi_2, fib_0, fib_1, nbehind, rho0, uwx, uwy)


def bounce_back_g(alpha, q, gi_0, gi_1, gib_0, nbehind, kappa, Tw):
    return lib().oracle_bounce_back_g(alpha, q, gi_0, gi_1, gib_0, nbehind, kappa, Tw)


def momentum_exchange(alpha, fi_post, fibar_new, uwx, uwy, rwx, rwy):
    o = _arr(3)
    lib().oracle_momentum_exchange(alpha, fi_post, fibar_new, uwx, uwy, rwx, rwy, _d(o))
    return o


def repulsion_mag(Cf, eps, s, delta, power):
    return lib().oracle_repulsion_mag(Cf, eps, s, delta, power)


def integrate(state6, Fx, Fy, Tz, mass, inertia):
    s = np.array(state6, dtype=np.float64)
    lib().oracle_integrate(_d(s), Fx, Fy, Tz, mass, inertia)
    return s


def refill_direction(nx_, ny_):
    return lib().oracle_refill_direction(nx_, ny_)


def ellipse_normal(dx, dy, a, b, c, s):
    nx_, ny_ = C.c_double(), C.c_double()
    lib().oracle_ellipse_normal(dx, dy, a, b, c, s, C.byref(nx_), C.byref(ny_))
    return nx_.value, ny_.value


def refill_f(nvalid, f1, f2, f3, rho0, uwx, uwy):
    f1 = np.ascontiguousarray(f1, dtype=np.float64)
    f2 = np.ascontiguousarray(f2, dtype=np.float64)
    f3 = np.ascontiguousarray(f3, dtype=np.float64)
    o = _arr(9)
    lib().oracle_refill_f(nvalid, _d(f1), _d(f2), _d(f3), rho0, uwx, uwy, _d(o))
    return o


# ---- whole simulation ---------------------------------------------------------------------
class OracleError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"oracle error {code}: {msg}")
        self.code = code


class OracleSim:
    def __init__(self, nx, ny, params):
        self.nx, self.ny, self.n = nx, ny, nx * ny
        self.params = dict(params)
        self._P = OracleParams.from_dict(params)
        self._h = C.c_void_p()
        rc = lib().oracle_create(nx, ny, C.byref(self._P), C.byref(self._h))
        if rc:
            raise OracleError(rc, lib().oracle_last_error(None).decode())

    @classmethod
    def from_workload(cls, w):
        sim = cls(w.nx, w.ny, w.params)
        if w.T_init is not None:
            sim.set_temperature(w.T_init)
        if w.particles is not None:
            sim.add_particles(**w.particles)
        return sim

    def _chk(self, rc):
        if rc:
            raise OracleError(rc, lib().oracle_last_error(self._h).decode())

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_temperature(self, T):
        T = np.ascontiguousarray(T, dtype=np.float64).reshape(-1)
        assert T.size == self.n
        self._chk(lib().oracle_set_temperature(self._h, _d(T)))

    def add_particles(self, x, y, diam, rho_ratio, T_w, ux=None, uy=None, omega=None, fixed=None,
                      minor=None, theta=None):
        """Circles of diameter `diam`; with `minor` and `theta`: ellipses of full axes diam x minor,
        the `diam` axis at angle theta to x."""
        c = lambda a: None if a is None else np.ascontiguousarray(a, dtype=np.float64)  # noqa: E731
        x, y, diam, rho_ratio, T_w, ux, uy, omega = map(c, (x, y, diam, rho_ratio, T_w, ux, uy, omega))
        fx = None if fixed is None else np.ascontiguousarray(fixed, dtype=np.uint8)
        if minor is not None:
            minor = c(minor)
            theta = c(np.zeros_like(x) if theta is None else theta)
            self._chk(lib().oracle_add_ellipses(
                self._h, int(x.size), _d(x), _d(y), _d(diam), _d(minor), _d(theta), _d(rho_ratio),
                _d(T_w), _d(ux), _d(uy), _d(omega), None if fx is None else fx.ctypes.data_as(_bp)))
            return
        self._chk(lib().oracle_add_particles(
            self._h, int(x.size), _d(x), _d(y), _d(diam), _d(rho_ratio), _d(T_w), _d(ux), _d(uy),
            _d(omega), None if fx is None else fx.ctypes.data_as(_bp)))

    def step(self, nsteps=1):
        self._chk(lib().oracle_step(self._h, int(nsteps)))

    def fields(self, populations=False):
        n = self.n
        out = {k: _arr(n) for k in ("rho", "ux", "uy", "T")}
        f = _arr(9 * n) if populations else None
        g = _arr(5 * n) if populations else None
        flag = np.empty(n, dtype=np.uint8)
        self._chk(lib().oracle_get_fields(self._h, _d(out["rho"]), _d(out["ux"]), _d(out["uy"]),
                                          _d(out["T"]), _d(f), _d(g), flag.ctypes.data_as(_bp)))
        res = {k: v.reshape(self.ny, self.nx) for k, v in out.items()}
        res["flag"] = flag.reshape(self.ny, self.nx)
        if populations:
            res["f"] = f.reshape(9, self.ny, self.nx)
            res["g"] = g.reshape(5, self.ny, self.nx)
        return res

    def set_state(self, f_post, g_post, particles):
        """Inject post-collision populations (9, ny, nx), (5, ny, nx) and a particle-state dict
        (x, y, theta, ux, uy, omega); the next step() starts after the collision."""
        f = np.ascontiguousarray(f_post, dtype=np.float64).reshape(-1)
        g = np.ascontiguousarray(g_post, dtype=np.float64).reshape(-1)
        assert f.size == 9 * self.n and g.size == 5 * self.n
        P = {k: np.ascontiguousarray(particles[k], dtype=np.float64)
             for k in ("x", "y", "theta", "ux", "uy", "omega")}
        self._chk(lib().oracle_set_state(self._h, _d(f), _d(g), int(P["x"].size),
                                         *[_d(P[k]) for k in ("x", "y", "theta", "ux", "uy", "omega")]))

    def precollision(self):
        f, g = _arr(9 * self.n), _arr(5 * self.n)
        self._chk(lib().oracle_get_precollision(self._h, _d(f), _d(g)))
        return f.reshape(9, self.ny, self.nx), g.reshape(5, self.ny, self.nx)

    def particles(self):
        n = C.c_int()
        self._chk(lib().oracle_get_particles(self._h, C.byref(n), *([None] * 9)))
        names = ("x", "y", "theta", "ux", "uy", "omega", "Fx", "Fy", "Tz")
        out = {k: _arr(n.value) for k in names}
        self._chk(lib().oracle_get_particles(self._h, C.byref(n), *[_d(out[k]) for k in names]))
        return out

    def _links(self, fn):
        n = C.c_longlong(0)
        rc = fn(self._h, C.byref(n), None, None, None, None, None)
        if rc not in (0, -3):
            self._chk(rc)
        m = n.value
        pid, i, j, al = (np.empty(m, dtype=np.int32) for _ in range(4))
        q = _arr(m)
        n = C.c_longlong(m)
        self._chk(fn(self._h, C.byref(n), pid.ctypes.data_as(_ip), i.ctypes.data_as(_ip),
                     j.ctypes.data_as(_ip), al.ctypes.data_as(_ip), _d(q)))
        return dict(pid=pid, i=i, j=j, alpha=al, q=q)

    def links(self):
        return self._links(lib().oracle_get_links)

    def links_bruteforce(self):
        return self._links(lib().oracle_get_links_bruteforce)
