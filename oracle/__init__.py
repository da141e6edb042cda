"""ctypes binding of the CPU oracle (oracle/oracle.c).  TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It does not import paper_2603_24508_b200 and shares no code with
the CUDA path.  All arrays are numpy, host memory, modified in place where the C routine
does so.
"""
import ctypes as C

import numpy as np

from . import build as _build

PERIODIC = 0
ABSORBING = 1

_lib = None
_lib_omp = None


def lib_omp():
    """The threaded twin (oracle/oracle_omp.c): same results as lib(), bit for bit, on all host cores."""
    global _lib_omp
    if _lib_omp is None:
        _lib_omp = C.CDLL(_build.build_omp())
        dp, ip, u64p = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_uint64)
        i64p = C.POINTER(C.c_int64)
        _lib_omp.oracle_omp_max_threads.argtypes = []
        _lib_omp.oracle_omp_max_threads.restype = C.c_int
        _lib_omp.oracle_omp_push.argtypes = [C.c_int64, dp, dp, dp, dp, ip, C.c_int32, C.c_double, C.c_double,
                                             C.c_int32, dp, C.c_double, dp, u64p, C.c_int32]
        _lib_omp.oracle_omp_push.restype = C.c_int
        _lib_omp.oracle_omp_arrange.argtypes = [C.c_int64, dp, dp, dp, dp, ip, dp, dp, dp, dp, ip, C.c_int32, ip, ip,
                                                C.c_int32]
        _lib_omp.oracle_omp_arrange.restype = C.c_int64
        _lib_omp.oracle_omp_run.argtypes = [C.c_int32, C.c_int32, i64p, i64p, dp, dp, dp, dp, ip, dp, dp, dp, dp, ip,
                                            C.c_int32, C.c_double, C.c_double, C.c_int32, dp, C.c_double, dp, u64p,
                                            ip, ip, C.c_int32]
        _lib_omp.oracle_omp_run.restype = C.c_int
    return _lib_omp


def omp_max_threads():
    return int(lib_omp().oracle_omp_max_threads())


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        dp, ip, u64p = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_uint64)
        i64p = C.POINTER(C.c_int64)
        _lib.oracle_boris_constants.argtypes = [C.c_double, C.c_double, C.c_double, dp, dp]
        _lib.oracle_boris_constants.restype = None
        _lib.oracle_push.argtypes = [C.c_int64, dp, dp, dp, dp, ip, C.c_int32, C.c_double, C.c_double,
                                     C.c_int32, dp, C.c_double, dp, u64p]
        _lib.oracle_push.restype = C.c_int
        _lib.oracle_arrange.argtypes = [C.c_int64, dp, dp, dp, dp, ip, dp, dp, dp, dp, ip, C.c_int32, ip, ip]
        _lib.oracle_arrange.restype = C.c_int64
        _lib.oracle_run.argtypes = [C.c_int32, C.c_int32, i64p, i64p, dp, dp, dp, dp, ip, dp, dp, dp, dp, ip,
                                    C.c_int32, C.c_double, C.c_double, C.c_int32, dp, C.c_double, dp, u64p,
                                    ip, ip]
        _lib.oracle_run.restype = C.c_int
        _lib.oracle_deposit.argtypes = [C.c_int64, dp, ip, C.c_int32, C.c_double, C.c_int32, C.c_double, dp]
        _lib.oracle_deposit.restype = C.c_int
    return _lib


def _d(a):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    assert a.dtype == np.int32 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def boris_constants(qm, dt, dx, B):
    """-> dict h, t(3), s(3), inv_dx  (oracle_boris_constants)."""
    Bv = np.ascontiguousarray(B, dtype=np.float64)
    out = np.zeros(8)
    lib().oracle_boris_constants(qm, dt, dx, _d(Bv), _d(out))
    return {"h": out[0], "t": out[1:4].copy(), "s": out[4:7].copy(), "inv_dx": out[7]}


class State:
    """Host-side species state driven by the oracle: x, vx, vy, vz (f64), cell (i32), n."""

    def __init__(self, x, vx, vy, vz, cell, *, nc, dx, dt, boundary, E, qm, B, arrange_every=0, threads=None):
        """threads=None: the single-thread oracle (oracle.c, the authority).  threads=k >= 1 (0 = all cores):
        its threaded twin (oracle_omp.c), pinned bit-identical to it by tests/test_oracle_omp.py."""
        self.threads = threads
        self.cap = len(x)
        self.x = np.array(x, dtype=np.float64)
        self.vx = np.array(vx, dtype=np.float64)
        self.vy = np.array(vy, dtype=np.float64)
        self.vz = np.array(vz, dtype=np.float64)
        self.cell = np.array(cell, dtype=np.int32)
        self.n = self.cap
        self.nc, self.dx, self.dt, self.boundary, self.qm = int(nc), float(dx), float(dt), int(boundary), float(qm)
        self.E = np.ascontiguousarray(E, dtype=np.float64)
        assert self.E.shape == (self.nc + 1,)
        self.B = np.ascontiguousarray(B, dtype=np.float64)
        self.arrange_every = int(arrange_every)
        self.steps = 0
        self.wall = np.zeros(2, dtype=np.uint64)
        self.count = np.zeros(self.nc, dtype=np.int32)
        self.offset = np.zeros(self.nc + 1, dtype=np.int32)
        self._tmp = None

    def _tmpbufs(self):
        if self._tmp is None:
            self._tmp = [np.empty(self.cap), np.empty(self.cap), np.empty(self.cap), np.empty(self.cap),
                         np.empty(self.cap, dtype=np.int32)]
        return self._tmp

    def push(self, nsteps=1):
        """nsteps mover steps with the arrange_every rule (oracle_run)."""
        t = self._tmpbufs()
        steps = C.c_int64(self.steps)
        n = C.c_int64(self.n)
        args = (nsteps, self.arrange_every, C.byref(steps), C.byref(n),
                _d(self.x), _d(self.vx), _d(self.vy), _d(self.vz), _i(self.cell),
                _d(t[0]), _d(t[1]), _d(t[2]), _d(t[3]), _i(t[4]),
                self.nc, self.dx, self.dt, self.boundary, _d(self.E), self.qm, _d(self.B),
                self.wall.ctypes.data_as(C.POINTER(C.c_uint64)), _i(self.count), _i(self.offset))
        if self.threads is None:
            rc = lib().oracle_run(*args)
        else:
            rc = lib_omp().oracle_omp_run(*args, int(self.threads))
        if rc:
            raise RuntimeError(f"oracle_run failed rc={rc}")
        self.steps, self.n = steps.value, n.value

    def push_only(self):
        """one bare mover step, no arrange, over slots [0,n) (oracle_push)."""
        args = (self.n, _d(self.x), _d(self.vx), _d(self.vy), _d(self.vz), _i(self.cell),
                self.nc, self.dx, self.dt, self.boundary, _d(self.E), self.qm, _d(self.B),
                self.wall.ctypes.data_as(C.POINTER(C.c_uint64)))
        rc = lib().oracle_push(*args) if self.threads is None else lib_omp().oracle_omp_push(*args, int(self.threads))
        if rc:
            raise RuntimeError(f"oracle_push failed rc={rc}")
        self.steps += 1

    def arrange(self):
        """explicit arrange (oracle_arrange); does not touch the step counter."""
        t = self._tmpbufs()
        args = (self.n, _d(self.x), _d(self.vx), _d(self.vy), _d(self.vz), _i(self.cell),
                _d(t[0]), _d(t[1]), _d(t[2]), _d(t[3]), _i(t[4]), self.nc, _i(self.count), _i(self.offset))
        nl = lib().oracle_arrange(*args) if self.threads is None else lib_omp().oracle_omp_arrange(*args, int(self.threads))
        if nl < 0:
            raise RuntimeError("oracle_arrange failed")
        for dst, src in zip((self.x, self.vx, self.vy, self.vz, self.cell), t):
            dst[:nl] = src[:nl]
        self.n = int(nl)

    def deposit(self, weight=1.0):
        """charge density on the nc+1 nodes from the current state (oracle_deposit)."""
        return deposit(self.x[:self.n], self.cell[:self.n], self.nc, self.dx, self.boundary, weight)

    def live(self):
        """the five arrays over [0,n)."""
        n = self.n
        return self.x[:n], self.vx[:n], self.vy[:n], self.vz[:n], self.cell[:n]


def deposit(x, cell, nc, dx, boundary, weight=1.0):
    """oracle_deposit -> rho on nc+1 nodes."""
    xa = np.ascontiguousarray(x, dtype=np.float64)
    ca = np.ascontiguousarray(cell, dtype=np.int32)
    rho = np.zeros(nc + 1)
    rc = lib().oracle_deposit(len(xa), _d(xa), _i(ca), int(nc), float(dx), int(boundary), float(weight), _d(rho))
    if rc:
        raise RuntimeError(f"oracle_deposit failed rc={rc}")
    return rho


def arrange_arrays(x, vx, vy, vz, cell, nc):
    """Pure function form of oracle_arrange -> (xo, vxo, vyo, vzo, cello, count, offset, n_live)."""
    n = len(x)
    a = [np.ascontiguousarray(v, dtype=np.float64) for v in (x, vx, vy, vz)]
    c = np.ascontiguousarray(cell, dtype=np.int32)
    o = [np.zeros(n) for _ in range(4)]
    co = np.full(n, -7, dtype=np.int32)
    count = np.zeros(nc, dtype=np.int32)
    offset = np.zeros(nc + 1, dtype=np.int32)
    nl = lib().oracle_arrange(n, _d(a[0]), _d(a[1]), _d(a[2]), _d(a[3]), _i(c), _d(o[0]), _d(o[1]), _d(o[2]),
                              _d(o[3]), _i(co), nc, _i(count), _i(offset))
    if nl < 0:
        raise RuntimeError("oracle_arrange failed")
    return o[0][:nl], o[1][:nl], o[2][:nl], o[3][:nl], co[:nl], count, offset, int(nl)


# ---- field solve (oracle/oracle_field.c): smoother, Poisson solve, E from phi -------------------------------------
_lib_field = None


def lib_field():
    global _lib_field
    if _lib_field is None:
        _lib_field = C.CDLL(_build.build_field())
        dp = C.POINTER(C.c_double)
        _lib_field.oracle_smooth.argtypes = [C.c_int32, C.c_int32, C.c_int32, dp, dp]
        _lib_field.oracle_poisson.argtypes = [C.c_int32, C.c_double, C.c_int32, dp, dp]
        _lib_field.oracle_efield.argtypes = [C.c_int32, C.c_double, C.c_int32, dp, dp]
        _lib_field.oracle_field_solve.argtypes = [C.c_int32, C.c_double, C.c_int32, C.c_int32, dp, dp, dp, dp]
        for f in (_lib_field.oracle_smooth, _lib_field.oracle_poisson, _lib_field.oracle_efield,
                  _lib_field.oracle_field_solve):
            f.restype = C.c_int
    return _lib_field


def _nodes(a, nc):
    a = np.ascontiguousarray(a, dtype=np.float64)
    assert a.shape == (nc + 1,)
    return a


def smooth(rho, nc, boundary, passes=1):
    """oracle_smooth -> filtered rho on nc+1 nodes."""
    out = np.zeros(nc + 1)
    rc = lib_field().oracle_smooth(int(nc), int(boundary), int(passes), _d(_nodes(rho, nc)), _d(out))
    if rc:
        raise RuntimeError(f"oracle_smooth failed rc={rc}")
    return out


def poisson(rho, nc, dx, boundary):
    """oracle_poisson -> phi on nc+1 nodes."""
    phi = np.zeros(nc + 1)
    rc = lib_field().oracle_poisson(int(nc), float(dx), int(boundary), _d(_nodes(rho, nc)), _d(phi))
    if rc:
        raise RuntimeError(f"oracle_poisson failed rc={rc}")
    return phi


def efield(phi, nc, dx, boundary):
    """oracle_efield -> E on nc+1 nodes."""
    E = np.zeros(nc + 1)
    rc = lib_field().oracle_efield(int(nc), float(dx), int(boundary), _d(_nodes(phi, nc)), _d(E))
    if rc:
        raise RuntimeError(f"oracle_efield failed rc={rc}")
    return E


def field_solve(rho, nc, dx, boundary, passes=0):
    """oracle_field_solve: smooth -> Poisson -> E.  -> (rho_smoothed, phi, E)."""
    rs, phi, E = np.zeros(nc + 1), np.zeros(nc + 1), np.zeros(nc + 1)
    rc = lib_field().oracle_field_solve(int(nc), float(dx), int(boundary), int(passes), _d(_nodes(rho, nc)), _d(rs),
                                        _d(phi), _d(E))
    if rc:
        raise RuntimeError(f"oracle_field_solve failed rc={rc}")
    return rs, phi, E
