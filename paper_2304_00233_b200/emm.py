"""Thin ctypes binding of libemm_b200.so (include/emm.h): argument marshalling only.

Every step of the method runs in the library's CUDA kernels; PyTorch is used here for device
memory (the workspace tensor) and the stream, as the ABI asks.  There is no CPU fallback: a
missing library or a missing CUDA device raises.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libemm_b200.so")
_SRC = [os.path.join(_HERE, "csrc", f) for f in ("emm_host.cu", "emm_kernels.cu", "emm_tile.cu", "emm_air.cu", "emm_air_sep.cu", "emm_air_cluster.cu", "emm_run.cu", "emm_sens.cu", "emm_noalloc.cu")]
_HDR = [os.path.join(_HERE, "csrc", f) for f in ("emm_internal.h", "emm_kernels.cuh", "emm_device.cuh")] + \
       [os.path.join(os.path.dirname(_HERE), "include", "emm.h")]

TOP_CPML, TOP_AIR = 0, 1
CHECK_CORNERS, CHECK_FACES, CHECK_FULL = 0, 1, 2
EINVAL, ENOMEM, ECUDA, ENOCONV, ENAN = -1, -2, -3, -4, -5
_GET = {"E1": 0, "E2": 1, "E3": 2, "H1": 3, "H2": 4, "H3": 5,
        "F_E1": 10, "F_E2": 11, "F_E3": 12, "F_H1": 13, "F_H2": 14, "F_H3": 15,
        "CE1": 20, "CE2": 21, "CE3": 22, "JW": 30, "DELTA": 31, "DTFT_GROUP": 32, "CHECK_N": 33, "CHECK_ACC": 34}
_INFO = ("N1", "N2", "N3", "lo1", "lo2", "lo3", "k0", "uniform_xy", "box_lo1", "box_lo2", "box_lo3",
         "box_hi1", "box_hi2", "box_hi3", "aux_M1", "aux_M2", "pitch", "air_cluster")
# every symbol include/emm.h declares (tests check that the library exports all of them)
SYMBOLS = ("emm_nugrid", "emm_fd_weights", "emm_dipole_direction", "emm_receiver_channels", "emm_grid_create", "emm_grid_destroy", "emm_grid_info", "emm_grid_coords",
           "emm_grid_fdcoef", "emm_workspace_bytes", "emm_bind_device", "emm_model_set", "emm_run", "emm_run_begin",
           "emm_run_steps", "emm_run_enqueue", "emm_run_end", "emm_get", "emm_profile", "emm_profile_read",
           "emm_launch_count", "emm_last_error", "emm_check_delta_static", "emm_sensitivity")


def build(force=False, verbose=False):
    """nvcc -> libemm_b200.so in-tree, sm_100a only."""
    deps = _SRC + _HDR
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= max(os.path.getmtime(p) for p in deps):
        return _SO
    cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-o", _SO] + _SRC + ["-lcufft", "-Xlinker", "-rpath=/usr/local/cuda/lib64"]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.check_call(cmd)
    return _SO


class GridOpts(C.Structure):
    _fields_ = [("rd", C.c_int), ("nb", C.c_int), ("ne", C.c_int), ("top", C.c_int),
                ("f0", C.c_double), ("cfl", C.c_double), ("aux_dx", C.c_double), ("air_route", C.c_int)]


class Src(C.Structure):
    _fields_ = [("pos", C.c_double * 3), ("dir", C.c_double * 3), ("type", C.c_int)]


class RunOpts(C.Structure):
    _fields_ = [("max_steps", C.c_int), ("fixed_steps", C.c_int), ("tol", C.c_double),
                ("check_every", C.c_int), ("check_set", C.c_int), ("fmax", C.c_double), ("batched", C.c_int),
                ("dtft_every", C.c_int), ("sparse_dft", C.c_int), ("dtft_pair", C.c_int)]


class EmmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libemm_b200 error %d: %s" % (code, msg))
        self.code = code


_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError("libemm_b200.so is not built (run __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(_SO)
        dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p
        L.emm_last_error.restype = C.c_char_p
        L.emm_nugrid.argtypes = [C.c_int, C.c_double, C.c_double, dp, dp]
        L.emm_fd_weights.argtypes = [C.c_int, dp, C.c_double, dp, dp]
        L.emm_dipole_direction.argtypes = [C.c_double, C.c_double, dp]
        L.emm_receiver_channels.argtypes = [dp, C.c_int, dp, dp, dp]
        L.emm_grid_create.argtypes = [dp, C.c_int, dp, C.c_int, dp, C.c_int, C.POINTER(GridOpts), C.POINTER(vp)]
        L.emm_grid_destroy.argtypes = [vp]
        L.emm_grid_destroy.restype = None
        L.emm_grid_info.argtypes = [vp, ip, dp]
        L.emm_grid_coords.argtypes = [vp, C.c_int, dp]
        L.emm_grid_fdcoef.argtypes = [vp, C.c_int, C.c_int, dp]
        L.emm_workspace_bytes.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
        L.emm_workspace_bytes.restype = C.c_size_t
        L.emm_bind_device.argtypes = [vp, vp, C.c_size_t, vp]
        L.emm_model_set.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.emm_run.argtypes = [vp, C.POINTER(Src), C.c_int, dp, C.c_int, dp, C.c_int, C.POINTER(RunOpts), dp, ip]
        L.emm_run_begin.argtypes = [vp, C.POINTER(Src), C.c_int, dp, C.c_int, dp, C.c_int, C.POINTER(RunOpts)]
        L.emm_run_steps.argtypes = [vp, C.c_int, ip, ip]
        L.emm_run_enqueue.argtypes = [vp, C.c_int]
        L.emm_run_end.argtypes = [vp, dp, ip]
        L.emm_get.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp]
        L.emm_sensitivity.argtypes = [vp, C.c_int, C.c_int, C.c_int, dp, dp]
        L.emm_profile.argtypes = [vp, C.c_int]
        L.emm_profile_read.argtypes = [vp, dp, ip]
        L.emm_check_delta_static.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp]
        L.emm_launch_count.argtypes = [vp]
        L.emm_launch_count.restype = C.c_longlong
        _lib = L
    return _lib


def _chk(rc, allow=()):
    if rc != 0 and rc not in allow:
        raise EmmError(rc, lib().emm_last_error().decode())
    return rc


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


CHECK_STATIC_MAX_NSRC = 16


def check_delta_static(acc_now, acc_prev, out=None, stream=None):
    """emm_check_delta_static: acc_now, acc_prev = CUDA torch tensors, complex128 [nsrc][6][nchk]; returns (or fills) a
    CUDA float64 tensor [nsrc][2].  Marshalling only: the library call allocates nothing; `out` lets the caller supply
    the output too (otherwise torch allocates those 16 * nsrc bytes here, outside the library)."""
    import torch
    assert acc_now.is_cuda and acc_prev.is_cuda and acc_now.dtype == acc_prev.dtype == torch.complex128
    assert acc_now.is_contiguous() and acc_prev.is_contiguous() and acc_now.shape == acc_prev.shape and acc_now.dim() == 3 and acc_now.shape[1] == 6
    nsrc, nchk = int(acc_now.shape[0]), int(acc_now.shape[2])
    if out is None:
        out = torch.empty((nsrc, 2), dtype=torch.float64, device=acc_now.device)
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= 2 * nsrc
    st = stream if stream is not None else torch.cuda.current_stream(acc_now.device)
    with torch.cuda.device(acc_now.device):
        _chk(lib().emm_check_delta_static(C.c_void_p(acc_now.data_ptr()), C.c_void_p(acc_prev.data_ptr()), nchk, nsrc,
                                          C.c_void_p(out.data_ptr()), C.c_void_p(st.cuda_stream)))
    return out


def emm_nugrid(n, length, dx):
    x = np.zeros(n + 1)
    q = C.c_double()
    _chk(lib().emm_nugrid(n, length, dx, _dptr(x), C.byref(q)))
    return x, q.value


def emm_fd_weights(nodes, x0):
    nodes = np.ascontiguousarray(nodes, dtype=np.float64)
    wi, wd = np.zeros(len(nodes)), np.zeros(len(nodes))
    _chk(lib().emm_fd_weights(len(nodes), _dptr(nodes), x0, _dptr(wi), _dptr(wd)))
    return wi, wd


def emm_dipole_direction(azimuth, dip):
    d = np.zeros(3)
    _chk(lib().emm_dipole_direction(float(azimuth), float(dip), _dptr(d)))
    return d


def emm_receiver_channels(g6, azimuth, dip):
    """g6: complex [nrec][6] (one source, one frequency of emm_run's output) -> complex [nrec][2] (E channel, H channel)"""
    g6 = np.ascontiguousarray(g6, dtype=np.complex128)
    n = g6.shape[0]
    assert g6.shape == (n, 6)
    az = np.ascontiguousarray(np.broadcast_to(np.asarray(azimuth, dtype=np.float64), (n,)))
    dp_ = np.ascontiguousarray(np.broadcast_to(np.asarray(dip, dtype=np.float64), (n,)))
    out = np.zeros((n, 2), dtype=np.complex128)
    _chk(lib().emm_receiver_channels(g6.ctypes.data_as(C.POINTER(C.c_double)), n, _dptr(az), _dptr(dp_),
                                     out.ctypes.data_as(C.POINTER(C.c_double))))
    return out


nugrid, fd_weights = emm_nugrid, emm_fd_weights     # same names as the oracle binding, for shared test helpers


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
                int(o.pop("batched", 0)), int(o.pop("dtft_every", 0)), int(o.pop("sparse_dft", 0)),
                int(o.pop("dtft_pair", 0)))
    if o:
        raise TypeError("unknown run options %s" % sorted(o))
    return r


class Grid:
    """emm_grid handle + the torch workspace it is bound to."""

    def __init__(self, x, y, z, rd, nb, ne=-1, top=TOP_CPML, f0=1.0, cfl=0.99, aux_dx=0.0, air_route=0):
        x, y, z = (np.ascontiguousarray(v, dtype=np.float64) for v in (x, y, z))
        o = GridOpts(rd, nb, ne, top, f0, cfl, aux_dx, air_route)
        h = C.c_void_p()
        _chk(lib().emm_grid_create(_dptr(x), len(x), _dptr(y), len(y), _dptr(z), len(z), C.byref(o), C.byref(h)))
        self._h = h
        self.ncell = (len(x) - 1, len(y) - 1, len(z) - 1)
        self.rd = rd
        self._ws = None
        self._plan = None
        self._model = None

    def close(self):
        if getattr(self, "_h", None):
            try:
                lib().emm_grid_destroy(self._h)
            except TypeError:          # interpreter shutdown: module globals are already gone
                pass
            self._h = None
        self._ws = None

    __del__ = close

    def info(self):
        ints = (C.c_int * len(_INFO))()
        dt = C.c_double()
        _chk(lib().emm_grid_info(self._h, ints, C.byref(dt)))
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
        _chk(lib().emm_grid_coords(self._h, axis, _dptr(out)))
        return out

    def fdcoef(self, axis, plus):
        n = self.info()["N%d" % (axis + 1)]
        out = np.zeros((n, 2 * self.rd))
        _chk(lib().emm_grid_fdcoef(self._h, axis, int(plus), _dptr(out)))
        return out

    # -- device memory and stream come from torch --
    def workspace_bytes(self, nsrc, nfreq, max_steps, nrec, dtft_pair=0):
        n = lib().emm_workspace_bytes(self._h, nsrc, nfreq, max_steps, nrec, dtft_pair)
        if n == 0:
            raise EmmError(ECUDA, lib().emm_last_error().decode())
        return n

    def bind(self, nsrc=1, nfreq=1, max_steps=0, nrec=64, device=None, ws_bytes=None, dtft_pair=0):
        """ws_bytes: bind a workspace of exactly this size instead of emm_workspace_bytes() (tests of the tight-memory paths)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libemm_b200 needs a CUDA device; there is no CPU fallback")
        device = device or getattr(self, "_device", None) or "cuda:0"
        self._device = device
        max_steps = max_steps or 100000
        plan = (nsrc, nfreq, max_steps, nrec)
        torch.cuda.set_device(device)
        n = int(ws_bytes) if ws_bytes is not None else self.workspace_bytes(nsrc, nfreq, max_steps, nrec, dtft_pair)
        if ws_bytes is None and self._ws is not None and n <= self._ws.numel():
            return
        self._fixed_ws = ws_bytes is not None          # an explicitly sized workspace is never regrown by _ensure
        self._ws = None
        self._ws = torch.empty(n, dtype=torch.uint8, device=device)
        torch.cuda.synchronize(device)
        if getattr(self, "stream", None) is None:
            # a torch stream of its own: the legacy default stream cannot be captured into CUDA graphs
            self.stream = torch.cuda.Stream(device=device)
        stream = self.stream.cuda_stream
        _chk(lib().emm_bind_device(self._h, C.c_void_p(self._ws.data_ptr()), n, C.c_void_p(stream)))
        self._plan = plan

    def model_set(self, sigma_h, sigma_v=None):
        sh = np.ascontiguousarray(sigma_h, dtype=np.float32)
        assert sh.shape == self.ncell[::-1], (sh.shape, self.ncell)
        sv = None if sigma_v is None else np.ascontiguousarray(sigma_v, dtype=np.float32)
        self._model = (sh, sv)
        if self._ws is None:
            self.bind()
        fp = C.POINTER(C.c_float)
        _chk(lib().emm_model_set(self._h, sh.ctypes.data_as(fp), None if sv is None else sv.ctypes.data_as(fp)))

    def _ensure(self, nsrc, nfreq, nrec, opts):
        """grow the workspace if this run needs more than what is bound (re-uploads the model)"""
        o = opts or {}
        steps = int(o.get("fixed_steps", 0)) or int(o.get("max_steps", 0)) or 100000
        resident = nsrc if (o.get("batched", 0) or o.get("_resident", 0)) else 1
        plan = (resident, nfreq, steps, max(nrec, 1))
        if getattr(self, "_fixed_ws", False):
            return
        ws = self._ws
        self.bind(*[max(a, b) for a, b in zip(plan, self._plan or plan)], dtft_pair=int(o.get("dtft_pair", 0)))
        if self._ws is not ws and getattr(self, "_model", None) is not None:      # a larger workspace was bound: the model goes up again
            self.model_set(*self._model)

    def run(self, sources, freqs, receivers, opts=None, allow_noconv=False):
        freqs = np.ascontiguousarray(freqs, dtype=np.float64)
        rec = np.ascontiguousarray(receivers, dtype=np.float64).reshape(-1, 3)
        self._ensure(len(sources), len(freqs), len(rec), opts)
        out = np.zeros((len(sources), len(freqs), len(rec), 6), dtype=np.complex128)
        ns = np.zeros(len(sources), dtype=np.int32)
        o = _ropts(opts)
        self.last_rc = _chk(lib().emm_run(self._h, _srcs(sources), len(sources), _dptr(freqs), len(freqs), _dptr(rec), len(rec),
                                          C.byref(o), out.ctypes.data_as(C.POINTER(C.c_double)),
                                          ns.ctypes.data_as(C.POINTER(C.c_int))), allow=(ENOCONV,) if allow_noconv else ())
        return out, ns

    def run_begin(self, sources, freqs, receivers, opts=None):
        freqs = np.ascontiguousarray(freqs, dtype=np.float64)
        rec = np.ascontiguousarray(receivers, dtype=np.float64).reshape(-1, 3)
        o2 = dict(opts or {})
        o2["_resident"] = 1
        self._ensure(len(sources), len(freqs), len(rec), o2)
        self._shape_out = (len(sources), len(freqs), len(rec), 6)
        o = _ropts(opts)
        _chk(lib().emm_run_begin(self._h, _srcs(sources), len(sources), _dptr(freqs), len(freqs), _dptr(rec), len(rec),
                                 C.byref(o)))

    def run_steps(self, n, allow_noconv=True):
        ns = np.zeros(self._shape_out[0], dtype=np.int32)
        done = C.c_int()
        _chk(lib().emm_run_steps(self._h, n, ns.ctypes.data_as(C.POINTER(C.c_int)), C.byref(done)),
             allow=(ENOCONV,) if allow_noconv else ())
        return ns, bool(done.value)

    def run_enqueue(self, n):
        _chk(lib().emm_run_enqueue(self._h, n))

    def run_end(self):
        out = np.zeros(self._shape_out, dtype=np.complex128)
        ns = np.zeros(self._shape_out[0], dtype=np.int32)
        _chk(lib().emm_run_end(self._h, out.ctypes.data_as(C.POINTER(C.c_double)), ns.ctypes.data_as(C.POINTER(C.c_int))))
        return out, ns

    def get(self, what, isrc=0, ifreq=0):
        code = _GET[what]
        if what == "JW":
            out = np.zeros(self._shape_out[1], dtype=np.complex128)
        elif what == "DELTA":
            out = np.zeros(2)
        elif what in ("DTFT_GROUP", "CHECK_N"):
            out = np.zeros(1, dtype=np.int32)
        elif what == "CHECK_ACC":
            out = np.zeros((6, int(self.get("CHECK_N")[0])), dtype=np.complex128)
        elif what.startswith("F_"):
            out = np.zeros(self.shape, dtype=np.complex64)
        else:
            out = np.zeros(self.shape, dtype=np.float32)
        _chk(lib().emm_get(self._h, isrc, code, ifreq, out.ctypes.data_as(C.c_void_p)))
        return out

    def sensitivity(self, isrc, iadj, ifreq):
        """(d/d sigma_h, d/d sigma_v) of the E-field datum of transmitter `isrc` and receiver dipole `iadj`, complex [nz][ny][nx]."""
        nx, ny, nz = self.ncell
        kh, kv = np.zeros((nz, ny, nx), dtype=np.complex128), np.zeros((nz, ny, nx), dtype=np.complex128)
        _chk(lib().emm_sensitivity(self._h, isrc, iadj, ifreq, kh.ctypes.data_as(C.POINTER(C.c_double)), kv.ctypes.data_as(C.POINTER(C.c_double))))
        return kh, kv

    def profile(self, enable=True):
        _chk(lib().emm_profile(self._h, int(enable)))

    def profile_read(self):
        """(summed ms, launches) per update-kernel instance: E/H = one DTFT term per step (or decimated), E0/H0 = the
        accumulator-free steps of a DTFT pair, E2/H2 = its two-term steps."""
        ms = np.zeros(6)
        cnt = np.zeros(6, dtype=np.int32)
        _chk(lib().emm_profile_read(self._h, _dptr(ms), cnt.ctypes.data_as(C.POINTER(C.c_int))))
        return {k: (float(ms[q]), int(cnt[q])) for q, k in enumerate(("E", "H", "E0", "H0", "E2", "H2"))}

    def launch_count(self):
        return int(lib().emm_launch_count(self._h))


# ---- multi-GPU: replicas only -------------------------------------------------------
def shard_sources(nsrc, rank, world):
    """Sources are independent problems (one source per MPI rank, no messages): source s runs on
    rank s mod world."""
    return list(range(rank, nsrc, world))


def run_replicated(grid, sources, freqs, receivers, opts=None, group=None):
    """Every rank runs its share of the sources on its own GPU through `grid.run`; the per-source results are
    gathered on the host (all_gather_object).  No collective touches the data path."""
    import torch.distributed as dist
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    mine = shard_sources(len(sources), rank, world)
    out, ns = (grid.run([sources[s] for s in mine], freqs, receivers, opts) if mine
               else (np.zeros((0, len(freqs), len(np.reshape(receivers, (-1, 3))), 6), np.complex128), np.zeros(0, np.int32)))
    parts = [None] * world
    if world > 1:
        dist.all_gather_object(parts, (mine, out, ns), group=group)
    else:
        parts = [(mine, out, ns)]
    full = np.zeros((len(sources),) + out.shape[1:], dtype=np.complex128)
    steps = np.zeros(len(sources), dtype=np.int32)
    for idx, o, n in parts:
        for q, s in enumerate(idx):
            full[s], steps[s] = o[q], n[q]
    return full, steps
