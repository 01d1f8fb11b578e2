"""Thin ctypes binding over the C ABI of include/lbm.h (argument marshalling only).

PyTorch supplies the device workspace (one uint8 tensor) and the CUDA stream; every step of the
hot path runs in the library's own sm_100a kernels.  There is NO CPU fallback: if the shared
library is missing or no CUDA device is present, constructing a `Simulation` raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblbm_b200.so")

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_bp = C.POINTER(C.c_ubyte)

LBM_OK, LBM_E_ARG, LBM_E_STATE, LBM_E_CAPACITY, LBM_E_CUDA, LBM_E_NONFINITE = 0, -1, -2, -3, -4, -5


class LbmParams(C.Structure):
    """Mirror of `lbm_params` in include/lbm.h."""
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


class LbmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"lbm error {code}: {msg}")
        self.code = code


_lib = None


def load_library():
    """dlopen the C-ABI library and declare its signatures.  Raises if it has not been built
    (`python -m paper_2308_16597_b200.build` or `__graft_entry__.build()`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build the CUDA library first "
                           "(python paper_2308_16597_b200/build.py); there is no CPU fallback")
    L = C.CDLL(LIB_PATH)
    vp, sz, ll = C.c_void_p, C.c_size_t, C.c_longlong
    P = C.POINTER(LbmParams)
    L.lbm_params_default.argtypes = [P]
    L.lbm_params_default.restype = None
    L.lbm_workspace_bytes.argtypes = [C.c_int, C.c_int, P]
    L.lbm_workspace_bytes.restype = sz
    L.lbm_create.argtypes = [C.c_int, C.c_int, P, vp, sz, vp, C.POINTER(vp)]
    L.lbm_set_temperature.argtypes = [vp, _dp]
    L.lbm_add_particles.argtypes = [vp, C.c_int, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _bp]
    L.lbm_add_ellipses.argtypes = [vp, C.c_int, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _bp]
    L.lbm_step.argtypes = [vp, C.c_int]
    L.lbm_prepare.argtypes = [vp, C.c_int]
    L.lbm_set_overlap.argtypes = [vp, C.c_int]
    L.lbm_set_two_step.argtypes = [vp, C.c_int]
    L.lbm_set_tma.argtypes = [vp, C.c_int]
    L.lbm_set_band_steps.argtypes = [vp, C.c_int]
    L.lbm_set_graph.argtypes = [vp, C.c_int]
    L.lbm_set_band.argtypes = [vp, C.c_int]
    L.lbm_get_band.argtypes = [vp, C.POINTER(C.c_int)]
    L.lbm_slab_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, P]
    L.lbm_slab_workspace_bytes.restype = sz
    L.lbm_create_slab.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, P, vp, sz, vp, C.POINTER(vp)]
    L.lbm_slab_forces.argtypes = [vp]
    L.lbm_slab_force_buffer.argtypes = [vp, C.POINTER(vp), C.POINTER(C.c_int)]
    L.lbm_slab_advance.argtypes = [vp]
    L.lbm_slab_check.argtypes = [vp]
    L.lbm_slab_halo_doubles.argtypes = [vp, C.POINTER(ll)]
    L.lbm_slab_pack.argtypes = [vp, C.c_int, vp]
    L.lbm_slab_unpack.argtypes = [vp, C.c_int, vp]
    L.lbm_slab_exchange_halos.argtypes = [C.POINTER(vp), C.c_int]
    L.lbm_slab_combine_forces.argtypes = [C.POINTER(vp), C.c_int]
    L.lbm_slab_link_peers.argtypes = [C.POINTER(vp), C.c_int]
    L.lbm_slab_fence.argtypes = [C.POINTER(vp), C.c_int]
    L.lbm_get_fields.argtypes = [vp, _dp, _dp, _dp, _dp, _dp, _dp, _bp]
    L.lbm_get_macroscopic_static.argtypes = [vp, _dp, _dp, _dp, _dp]
    L.lbm_get_particles.argtypes = [vp, _ip] + [_dp] * 9
    L.lbm_get_links.argtypes = [vp, C.POINTER(ll), _ip, _ip, _ip, _ip, _dp]
    L.lbm_profile_enable.argtypes = [vp, C.c_int]
    L.lbm_profile_kernels.argtypes = []
    L.lbm_profile_kernel_name.argtypes = [C.c_int]
    L.lbm_profile_kernel_name.restype = C.c_char_p
    L.lbm_profile_get.argtypes = [vp, C.c_int, _dp, C.POINTER(ll)]
    L.lbm_kernel_launches.argtypes = [vp]
    L.lbm_kernel_launches.restype = ll
    L.lbm_destroy.argtypes = [vp]
    L.lbm_last_error.argtypes = [vp]
    L.lbm_last_error.restype = C.c_char_p
    for name in ("lbm_create", "lbm_set_temperature", "lbm_add_particles", "lbm_add_ellipses", "lbm_step",
                 "lbm_get_fields", "lbm_get_particles", "lbm_get_links", "lbm_profile_enable",
                 "lbm_profile_kernels", "lbm_profile_get", "lbm_destroy", "lbm_set_overlap",
                 "lbm_set_two_step", "lbm_set_graph", "lbm_set_band", "lbm_get_band", "lbm_create_slab",
                 "lbm_slab_forces", "lbm_slab_force_buffer", "lbm_slab_advance", "lbm_slab_check",
                 "lbm_slab_halo_doubles", "lbm_slab_pack", "lbm_slab_unpack", "lbm_slab_exchange_halos",
                 "lbm_slab_combine_forces", "lbm_slab_link_peers", "lbm_slab_fence",
                 "lbm_get_macroscopic_static", "lbm_prepare", "lbm_set_tma", "lbm_set_band_steps"):
        getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _host(a, pinned_ok=True):
    """numpy view of a host buffer (numpy array or CPU torch tensor, e.g. pinned)."""
    if a is None:
        return None
    if hasattr(a, "numpy") and not isinstance(a, np.ndarray):
        a = a.numpy()
    return np.ascontiguousarray(a, dtype=np.float64)


class Simulation:
    """One particle-resolved thermal LBM simulation on one B200 (calls follow include/lbm.h)."""

    def __init__(self, nx, ny, params, device="cuda:0", stream=None, slab=None):
        """slab = (j0, j1, halo): a y-slab of the nx x ny cavity (include/lbm.h "y-slabs"): the handle
        stores the rows [j0 - halo, j1 + halo) clipped to the cavity and owns [j0, j1); `ny`, `n` and
        the arrays of fields() then refer to the OWN rows, `rows_stored` to what set_temperature takes."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the lattice Boltzmann hot path has no CPU fallback")
        self._torch = torch
        self._L = load_library()
        self.nx, self.ny, self.n = int(nx), int(ny), int(nx) * int(ny)
        self.ny_global, self.slab = int(ny), None
        self.params = dict(params)
        self._P = LbmParams.from_dict(params)
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        if slab is not None:
            j0, j1, halo = (int(v) for v in slab)
            self.slab = (j0, j1, halo)
            lo, hi = (0 if j0 == 0 else j0 - halo), (int(ny) if j1 == int(ny) else j1 + halo)
            self.rows_stored = (lo, hi)
            self.ny, self.n = j1 - j0, int(nx) * (j1 - j0)
            nbytes = self._L.lbm_slab_workspace_bytes(self.nx, self.ny_global, j0, j1, halo, C.byref(self._P))
        else:
            self.rows_stored = (0, int(ny))
            nbytes = self._L.lbm_workspace_bytes(self.nx, self.ny, C.byref(self._P))
        if nbytes == 0:
            raise LbmError(LBM_E_ARG, "lbm_workspace_bytes: bad size or parameter")
        self.workspace_bytes = int(nbytes)
        self._ws = torch.empty(int(nbytes) + 256, dtype=torch.uint8, device=self.device)
        base = (self._ws.data_ptr() + 255) // 256 * 256
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = C.c_void_p()
        if slab is not None:
            rc = self._L.lbm_create_slab(self.nx, self.ny_global, j0, j1, halo, C.byref(self._P),
                                         C.c_void_p(base), C.c_size_t(int(nbytes)),
                                         C.c_void_p(self.stream.cuda_stream), C.byref(self._h))
        else:
            rc = self._L.lbm_create(self.nx, self.ny, C.byref(self._P), C.c_void_p(base),
                                    C.c_size_t(int(nbytes)), C.c_void_p(self.stream.cuda_stream),
                                    C.byref(self._h))
        if rc:
            raise LbmError(rc, self._L.lbm_last_error(None).decode())

    @classmethod
    def from_workload(cls, w, **kw):
        sim = cls(w.nx, w.ny, w.params, **kw)
        if w.T_init is not None:
            sim.set_temperature(w.T_init)
        if w.particles is not None:
            sim.add_particles(**w.particles)
        return sim

    def _chk(self, rc):
        if rc:
            raise LbmError(rc, self._L.lbm_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) and self._h:
            self._L.lbm_destroy(self._h)
            self._h = C.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- set-up ----
    def set_temperature(self, T):
        T = _host(T).reshape(-1)
        assert T.size == self.nx * (self.rows_stored[1] - self.rows_stored[0])
        self._chk(self._L.lbm_set_temperature(self._h, _d(T)))

    def add_particles(self, x, y, diam, rho_ratio, T_w, ux=None, uy=None, omega=None, fixed=None,
                      minor=None, theta=None):
        """lbm_add_particles; with `minor` (and `theta`): lbm_add_ellipses, full axes diam x minor,
        the `diam` axis at angle theta to x."""
        x, y, diam, rho_ratio, T_w, ux, uy, omega = map(_host, (x, y, diam, rho_ratio, T_w, ux, uy, omega))
        fx = None if fixed is None else np.ascontiguousarray(fixed, dtype=np.uint8)
        if minor is not None:
            minor = _host(minor)
            theta = _host(np.zeros_like(x) if theta is None else theta)
            self._chk(self._L.lbm_add_ellipses(
                self._h, int(x.size), _d(x), _d(y), _d(diam), _d(minor), _d(theta), _d(rho_ratio),
                _d(T_w), _d(ux), _d(uy), _d(omega), None if fx is None else fx.ctypes.data_as(_bp)))
            return
        self._chk(self._L.lbm_add_particles(
            self._h, int(x.size), _d(x), _d(y), _d(diam), _d(rho_ratio), _d(T_w), _d(ux), _d(uy),
            _d(omega), None if fx is None else fx.ctypes.data_as(_bp)))

    # ---- the hot path ----
    def step(self, nsteps=1):
        self._chk(self._L.lbm_step(self._h, int(nsteps)))

    def prepare(self, nsteps):
        """lbm_prepare: plans, captures and uploads what step(nsteps) will replay, without stepping."""
        self._chk(self._L.lbm_prepare(self._h, int(nsteps)))

    def set_overlap(self, on=True):
        self._chk(self._L.lbm_set_overlap(self._h, 1 if on else 0))

    def set_graph(self, on=True):
        self._chk(self._L.lbm_set_graph(self._h, 1 if on else 0))

    def set_band(self, on=True):
        """False / 0: off; True / 1: where it pays (bands of >= 2^18 nodes); 2: every band."""
        self._chk(self._L.lbm_set_band(self._h, int(on)))

    def band_rows(self):
        """Q of the last band plan: > 0: rows [0, Q) advance two steps per pass; < 0: rows [-Q, ny)
        (a band above the suspension); 0: none."""
        q = C.c_int(0)
        self._chk(self._L.lbm_get_band(self._h, C.byref(q)))
        return q.value

    def set_two_step(self, on=True):
        """Particle-free lattices: time steps per pass over the populations.  False / 0: one;
        True / 1 / 2: two; 3: three (lbm_set_two_step)."""
        self._chk(self._L.lbm_set_two_step(self._h, int(on)))

    def set_band_steps(self, steps):
        """Time steps per pass in a band under the suspension: 3 (default) or 2 (lbm_set_band_steps)."""
        self._chk(self._L.lbm_set_band_steps(self._h, int(steps)))

    def set_tma(self, on=True):
        """Three-step passes of a particle-free closed cavity: 0 / False the plain three-step kernel,
        1 / True the persistent TMA-fed kernel with group barriers, 2 the same with the row-wise
        hand-over (the default from 2^20 nodes) (lbm_set_tma)."""
        self._chk(self._L.lbm_set_tma(self._h, int(on)))

    # ---- y-slabs: the two halves of a step and the exchanges' end points (slabs.py drives them) ----
    def slab_forces(self):
        self._chk(self._L.lbm_slab_forces(self._h))

    def slab_advance(self):
        self._chk(self._L.lbm_slab_advance(self._h))

    def slab_check(self):
        self._chk(self._L.lbm_slab_check(self._h))

    def slab_force_tensor(self):
        """The slab's force buffer (3 * n doubles on the device) as a torch view of the workspace."""
        ptr, cnt = C.c_void_p(), C.c_int()
        self._chk(self._L.lbm_slab_force_buffer(self._h, C.byref(ptr), C.byref(cnt)))
        off = (ptr.value or 0) - self._ws.data_ptr()
        return self._ws[off:off + 8 * cnt.value].view(self._torch.float64)

    def slab_halo_doubles(self):
        n = C.c_longlong()
        self._chk(self._L.lbm_slab_halo_doubles(self._h, C.byref(n)))
        return n.value

    def slab_pack(self, side, buf):
        self._chk(self._L.lbm_slab_pack(self._h, int(side), C.c_void_p(buf.data_ptr())))

    def slab_unpack(self, side, buf):
        self._chk(self._L.lbm_slab_unpack(self._h, int(side), C.c_void_p(buf.data_ptr())))

    # ---- read-out ----
    def fields(self, populations=False, out=None):
        """dict of (ny, nx) arrays rho, ux, uy, T, flag (+ f (9,ny,nx), g (5,ny,nx) post-collision).
        `out` may supply preallocated host buffers (e.g. pinned torch tensors) by the same keys."""
        n = self.n
        out = out or {}
        bufs = {}
        for k in ("rho", "ux", "uy", "T"):
            b = out.get(k)
            bufs[k] = (b.numpy() if hasattr(b, "numpy") and not isinstance(b, np.ndarray) else b) \
                if b is not None else np.empty(n, dtype=np.float64)
        f = np.empty(9 * n, dtype=np.float64) if populations else None
        g = np.empty(5 * n, dtype=np.float64) if populations else None
        flag = np.empty(n, dtype=np.uint8)
        self._chk(self._L.lbm_get_fields(self._h, _d(bufs["rho"]), _d(bufs["ux"]), _d(bufs["uy"]),
                                         _d(bufs["T"]), _d(f), _d(g), flag.ctypes.data_as(_bp)))
        res = {k: v.reshape(self.ny, self.nx) for k, v in bufs.items()}
        res["flag"] = flag.reshape(self.ny, self.nx)
        if populations:
            res["f"] = f.reshape(9, self.ny, self.nx)
            res["g"] = g.reshape(5, self.ny, self.nx)
        return res

    def macroscopic_static(self):
        """rho, ux, uy, T through lbm_get_macroscopic_static (no allocation on the device, workspace
        untouched; lattices of at most 2^20 nodes)."""
        out = {k: np.empty(self.n, dtype=np.float64) for k in ("rho", "ux", "uy", "T")}
        self._chk(self._L.lbm_get_macroscopic_static(self._h, _d(out["rho"]), _d(out["ux"]),
                                                     _d(out["uy"]), _d(out["T"])))
        return {k: v.reshape(self.ny, self.nx) for k, v in out.items()}

    def particles(self):
        n = C.c_int()
        self._chk(self._L.lbm_get_particles(self._h, C.byref(n), *([None] * 9)))
        names = ("x", "y", "theta", "ux", "uy", "omega", "Fx", "Fy", "Tz")
        out = {k: np.empty(n.value, dtype=np.float64) for k in names}
        if n.value:
            self._chk(self._L.lbm_get_particles(self._h, C.byref(n), *[_d(out[k]) for k in names]))
        return out

    def links(self):
        n = C.c_longlong(0)
        rc = self._L.lbm_get_links(self._h, C.byref(n), None, None, None, None, None)
        if rc not in (LBM_OK, LBM_E_CAPACITY):
            self._chk(rc)
        m = n.value
        pid, i, j, al = (np.empty(m, dtype=np.int32) for _ in range(4))
        q = np.empty(m, dtype=np.float64)
        n = C.c_longlong(m)
        self._chk(self._L.lbm_get_links(self._h, C.byref(n), pid.ctypes.data_as(_ip),
                                        i.ctypes.data_as(_ip), j.ctypes.data_as(_ip),
                                        al.ctypes.data_as(_ip), _d(q)))
        return dict(pid=pid, i=i, j=j, alpha=al, q=q)

    # ---- profiling ----
    def kernel_launches(self):
        return int(self._L.lbm_kernel_launches(self._h))

    def profile(self, on=True):
        self._chk(self._L.lbm_profile_enable(self._h, 1 if on else 0))

    def profile_results(self):
        """{kernel name: (total ms over the sampled launches, number of sampled launches)}"""
        out = {}
        for k in range(self._L.lbm_profile_kernels()):
            ms, cnt = C.c_double(), C.c_longlong()
            self._chk(self._L.lbm_profile_get(self._h, k, C.byref(ms), C.byref(cnt)))
            out[self._L.lbm_profile_kernel_name(k).decode()] = (ms.value, cnt.value)
        return out
