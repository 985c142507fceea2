"""ctypes binding of oracle/libemm_oracle.so -- TEST INFRASTRUCTURE, NOT PRODUCT.

Argument marshalling only; every number is produced by oracle/emm_oracle.c.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libemm_oracle.so")

TOP_CPML, TOP_AIR = 0, 1
CHECK_CORNERS, CHECK_FACES, CHECK_FULL = 0, 1, 2
EINVAL, ENOMEM, ENOCONV, ENAN = -1, -2, -4, -5
COMPONENTS = ("E1", "E2", "E3", "H1", "H2", "H3")
_GET = {"E1": 0, "E2": 1, "E3": 2, "H1": 3, "H2": 4, "H3": 5,
        "F_E1": 10, "F_E2": 11, "F_E3": 12, "F_H1": 13, "F_H2": 14, "F_H3": 15,
        "CE1": 20, "CE2": 21, "CE3": 22, "JW": 30, "DELTA": 31, "CPML": 40}
_INFO = ("N1", "N2", "N3", "lo1", "lo2", "lo3", "k0", "uniform_xy", "box_lo1", "box_lo2", "box_lo3",
         "box_hi1", "box_hi2", "box_hi3", "aux_M1", "aux_M2")


def build(force=False):
    """Compile the oracle with gcc (plain -O2, OpenMP only spreads outer loops)."""
    src = os.path.join(_HERE, "emm_oracle.c")
    hdr = os.path.join(_HERE, "emm_oracle.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=gnu11", "-o", _SO, src, "-lm"])
    return _SO


class GridOpts(C.Structure):
    _fields_ = [("rd", C.c_int), ("nb", C.c_int), ("ne", C.c_int), ("top", C.c_int),
                ("f0", C.c_double), ("cfl", C.c_double), ("aux_dx", C.c_double)]


class Src(C.Structure):
    _fields_ = [("pos", C.c_double * 3), ("dir", C.c_double * 3), ("type", C.c_int)]


class RunOpts(C.Structure):
    _fields_ = [("max_steps", C.c_int), ("fixed_steps", C.c_int), ("tol", C.c_double),
                ("check_every", C.c_int), ("check_set", C.c_int), ("fmax", C.c_double),
                ("sparse_dft", C.c_int), ("dtft_every", C.c_int)]


class OracleError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("oracle error %d: %s" % (code, msg))
        self.code = code


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.emmo_last_error.restype = C.c_char_p
        dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p
        L.emmo_nugrid.argtypes = [C.c_int, C.c_double, C.c_double, dp, dp]
        L.emmo_fd_weights.argtypes = [C.c_int, dp, C.c_double, dp, dp]
        L.emmo_fft2.argtypes = [dp, C.c_int, C.c_int, C.c_int]
        L.emmo_grid_create.argtypes = [dp, C.c_int, dp, C.c_int, dp, C.c_int, C.POINTER(GridOpts), C.POINTER(vp)]
        L.emmo_grid_destroy.argtypes = [vp]
        L.emmo_grid_destroy.restype = None
        L.emmo_grid_info.argtypes = [vp, ip, dp]
        L.emmo_grid_coords.argtypes = [vp, C.c_int, dp]
        L.emmo_grid_fdcoef.argtypes = [vp, C.c_int, C.c_int, dp]
        L.emmo_model_set.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.emmo_run.argtypes = [vp, C.POINTER(Src), C.c_int, dp, C.c_int, dp, C.c_int, C.POINTER(RunOpts), dp, ip]
        L.emmo_run_begin.argtypes = [vp, C.POINTER(Src), C.c_int, dp, C.c_int, dp, C.c_int, C.POINTER(RunOpts)]
        L.emmo_run_steps.argtypes = [vp, C.c_int, ip, ip]
        L.emmo_run_end.argtypes = [vp, dp, ip]
        L.emmo_get.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp]
        L.emmo_sensitivity.argtypes = [vp, C.c_int, C.c_int, C.c_int, dp, dp]
        _lib = L
    return _lib


def _chk(rc, allow=()):
    if rc != 0 and rc not in allow:
        raise OracleError(rc, lib().emmo_last_error().decode())
    return rc


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def nugrid(n, length, dx):
    x = np.zeros(n + 1)
    q = C.c_double()
    _chk(lib().emmo_nugrid(n, length, dx, _dptr(x), C.byref(q)))
    return x, q.value


def fd_weights(nodes, x0):
    nodes = np.ascontiguousarray(nodes, dtype=np.float64)
    wi, wd = np.zeros(len(nodes)), np.zeros(len(nodes))
    _chk(lib().emmo_fd_weights(len(nodes), _dptr(nodes), x0, _dptr(wi), _dptr(wd)))
    return wi, wd


def fft2(a, sign):
    a = np.array(a, dtype=np.complex128, order="C")
    n2, n1 = a.shape
    _chk(lib().emmo_fft2(a.ctypes.data_as(C.POINTER(C.c_double)), n1, n2, sign))
    return a


def _srcs(sources):
    arr = (Src * len(sources))()
    for s, src in zip(arr, sources):       # (pos, dir) = electric dipole; (pos, dir, "M") = magnetic dipole
        s.pos[:] = [float(v) for v in src[0]]
        s.dir[:] = [float(v) for v in src[1]]
        s.type = 1 if len(src) > 2 and str(src[2]).upper().startswith("M") else 0
    return arr


def _ropts(o):
    o = dict(o or {})
    r = RunOpts(int(o.pop("max_steps", 0)), int(o.pop("fixed_steps", 0)), float(o.pop("tol", 0)),
                int(o.pop("check_every", 0)), int(o.pop("check_set", CHECK_FACES)), float(o.pop("fmax", 0)),
                int(o.pop("sparse_dft", 0)), int(o.pop("dtft_every", 0)))
    o.pop("batched", None)
    if o:
        raise TypeError("unknown run options %s" % sorted(o))
    return r


class Grid:
    def __init__(self, x, y, z, rd, nb, ne=-1, top=TOP_CPML, f0=1.0, cfl=0.99, aux_dx=0.0):
        x, y, z = (np.ascontiguousarray(v, dtype=np.float64) for v in (x, y, z))
        o = GridOpts(rd, nb, ne, top, f0, cfl, aux_dx)
        h = C.c_void_p()
        _chk(lib().emmo_grid_create(_dptr(x), len(x), _dptr(y), len(y), _dptr(z), len(z), C.byref(o), C.byref(h)))
        self._h = h
        self.ncell = (len(x) - 1, len(y) - 1, len(z) - 1)
        self.rd = rd
        self.nb = nb

    def close(self):
        if getattr(self, "_h", None):
            try:
                lib().emmo_grid_destroy(self._h)
            except TypeError:          # interpreter shutdown: module globals are already gone
                pass
            self._h = None

    __del__ = close

    def info(self):
        ints = (C.c_int * len(_INFO))()
        dt = C.c_double()
        _chk(lib().emmo_grid_info(self._h, ints, C.byref(dt)))
        d = dict(zip(_INFO, list(ints)))
        d["dt"] = dt.value
        return d

    @property
    def shape(self):
        i = self.info()
        return (i["N3"], i["N2"], i["N1"])

    def coords(self, axis):
        n = self.info()["N%d" % (axis + 1)]
        out = np.zeros(n + 1)
        _chk(lib().emmo_grid_coords(self._h, axis, _dptr(out)))
        return out

    def fdcoef(self, axis, plus):
        n = self.info()["N%d" % (axis + 1)]
        out = np.zeros((n, 2 * self.rd))
        _chk(lib().emmo_grid_fdcoef(self._h, axis, int(plus), _dptr(out)))
        return out

    def model_set(self, sigma_h, sigma_v=None):
        sh = np.ascontiguousarray(sigma_h, dtype=np.float32)
        assert sh.shape == self.ncell[::-1], (sh.shape, self.ncell)
        fp = C.POINTER(C.c_float)
        sv = None if sigma_v is None else np.ascontiguousarray(sigma_v, dtype=np.float32)
        _chk(lib().emmo_model_set(self._h, sh.ctypes.data_as(fp), None if sv is None else sv.ctypes.data_as(fp)))

    def run(self, sources, freqs, receivers, opts=None, allow_noconv=False):
        freqs = np.ascontiguousarray(freqs, dtype=np.float64)
        rec = np.ascontiguousarray(receivers, dtype=np.float64).reshape(-1, 3)
        out = np.zeros((len(sources), len(freqs), len(rec), 6), dtype=np.complex128)
        ns = np.zeros(len(sources), dtype=np.int32)
        o = _ropts(opts)
        rc = _chk(lib().emmo_run(self._h, _srcs(sources), len(sources), _dptr(freqs), len(freqs), _dptr(rec), len(rec),
                                 C.byref(o), out.ctypes.data_as(C.POINTER(C.c_double)),
                                 ns.ctypes.data_as(C.POINTER(C.c_int))), allow=(ENOCONV,) if allow_noconv else ())
        self.last_rc = rc
        return out, ns

    def run_begin(self, sources, freqs, receivers, opts=None):
        freqs = np.ascontiguousarray(freqs, dtype=np.float64)
        rec = np.ascontiguousarray(receivers, dtype=np.float64).reshape(-1, 3)
        self._shape_out = (len(sources), len(freqs), len(rec), 6)
        o = _ropts(opts)
        _chk(lib().emmo_run_begin(self._h, _srcs(sources), len(sources), _dptr(freqs), len(freqs), _dptr(rec), len(rec),
                                  C.byref(o)))

    def run_steps(self, n, allow_noconv=True):
        ns = np.zeros(self._shape_out[0], dtype=np.int32)
        done = C.c_int()
        _chk(lib().emmo_run_steps(self._h, n, ns.ctypes.data_as(C.POINTER(C.c_int)), C.byref(done)),
             allow=(ENOCONV,) if allow_noconv else ())
        return ns, bool(done.value)

    def run_end(self):
        out = np.zeros(self._shape_out, dtype=np.complex128)
        ns = np.zeros(self._shape_out[0], dtype=np.int32)
        _chk(lib().emmo_run_end(self._h, out.ctypes.data_as(C.POINTER(C.c_double)), ns.ctypes.data_as(C.POINTER(C.c_int))))
        return out, ns

    def sensitivity(self, isrc, iadj, ifreq):
        nx, ny, nz = self.ncell
        kh, kv = np.zeros((nz, ny, nx), dtype=np.complex128), np.zeros((nz, ny, nx), dtype=np.complex128)
        _chk(lib().emmo_sensitivity(self._h, isrc, iadj, ifreq, kh.ctypes.data_as(C.POINTER(C.c_double)), kv.ctypes.data_as(C.POINTER(C.c_double))))
        return kh, kv

    def get(self, what, isrc=0, ifreq=0):
        code = _GET[what]
        if what == "JW":
            out = np.zeros(self._shape_out[1], dtype=np.complex128)
        elif what == "DELTA":
            out = np.zeros(2)
        elif what == "CPML":                 # ifreq = axis; rows: a(node), b(node), a(half node), b(half node)
            out = np.zeros((4, 2 * self.nb))
        elif what.startswith("F_"):
            out = np.zeros(self.shape, dtype=np.complex128)
        else:
            out = np.zeros(self.shape)
        _chk(lib().emmo_get(self._h, isrc, code, ifreq, out.ctypes.data_as(C.c_void_p)))
        return out
