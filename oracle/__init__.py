"""CPU oracle for the collision-term hot path -- TEST INFRASTRUCTURE, not product code.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the CUDA package
``paper_2308_04869_b200`` and shares no code with it.

``rbg_oracle.cpp`` is the oracle proper (Eq. 16-19, chain O0..O14 of
DESIGN.md section 4); ``quadrature.py`` and ``eq37.py`` are independent evaluations of the same
integral used to pin it.  This module only builds the shared object and marshals arguments.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "rbg_oracle.cpp"
_LIB = _HERE / "librbg_oracle.so"


def _cpu_has_fma() -> bool:
    try:
        return " fma " in open("/proc/cpuinfo").read().replace("\n", " ")
    except OSError:
        return False


def build(force: bool = False) -> Path:
    """Compile the oracle with g++ (no CUDA).  -ffp-contract=off: every rounding is explicit.

    RBG_ORACLE_SANITIZE=1 in the environment builds and loads librbg_oracle_san.so instead, compiled with
    -fsanitize=address,undefined (run the CPU pins under it with LD_PRELOAD=$(gcc -print-file-name=libasan.so);
    profiles/r2_sanitizers.md has the command and its result)."""
    san = os.environ.get("RBG_ORACLE_SANITIZE", "") not in ("", "0")
    lib_path = _HERE / "librbg_oracle_san.so" if san else _LIB
    tag = _HERE / (".build_tag_san" if san else ".build_tag")
    want = f"fma={int(_cpu_has_fma())} mtime={_SRC.stat().st_mtime_ns}"
    if not force and lib_path.exists() and tag.exists() and tag.read_text() == want:
        return lib_path
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
           "-o", str(lib_path), str(_SRC)]
    if san:
        cmd[1:1] = ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
    if _cpu_has_fma():
        cmd.insert(1, "-mfma")          # std::fma -> one vfmadd instruction instead of a libm call
    subprocess.run(cmd, check=True)
    tag.write_text(want)
    return lib_path


class _Species(C.Structure):
    _fields_ = [("mass", C.c_double), ("charge", C.c_double), ("stat", C.c_int), ("g", C.c_double)]


class _Grid(C.Structure):
    _fields_ = [("n", C.c_int * 3), ("pmin", C.c_double * 3), ("pmax", C.c_double * 3)]


class _Process(C.Structure):
    _fields_ = [("a", C.c_int), ("b", C.c_int), ("c", C.c_int), ("d", C.c_int), ("kind", C.c_int),
                ("par", C.c_double * 4), ("sym", C.c_double), ("sampler", C.c_int)]


FCALLBACK = C.CFUNCTYPE(C.c_double, C.c_int, C.POINTER(C.c_double), C.c_void_p)

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_int, C.POINTER(_Species), C.POINTER(_Grid), C.c_int,
                                 C.POINTER(_Process), C.c_double, C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        for name in ("orc_f_elems", "orc_detail_elems"):
            getattr(L, name).restype = C.c_size_t
            getattr(L, name).argtypes = [C.c_void_p]
        L.orc_species_offset.restype = C.c_size_t
        L.orc_species_offset.argtypes = [C.c_void_p, C.c_int]
        L.orc_role_offset.restype = C.c_size_t
        L.orc_role_offset.argtypes = [C.c_void_p, C.c_int]
        L.orc_n_roles.argtypes = [C.c_void_p]
        L.orc_role_info.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int),
                                    C.POINTER(C.c_double), C.POINTER(C.c_int)]
        dp = C.POINTER(C.c_double)
        L.orc_collision.argtypes = [C.c_void_p, dp, dp, C.c_int, C.c_uint64, C.c_int, C.c_int, C.c_int,
                                    dp, dp, dp, dp, C.c_void_p, C.c_void_p, C.c_int]
        L.orc_collision_point.argtypes = [C.c_void_p, dp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_uint64,
                                          dp, C.c_void_p, C.c_void_p, C.c_int]
        L.orc_trace.argtypes = [C.c_void_p, dp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_uint64, dp,
                                C.POINTER(C.c_int), C.c_void_p, C.c_void_p, C.c_int]
        L.orc_collision_symmetric.argtypes = [C.c_void_p, dp, dp, dp, C.c_int, C.c_uint64, C.c_int, C.c_int, C.c_int, C.c_int]
        L.orc_m2_qcd.restype = C.c_double
        L.orc_m2_qcd.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double]
        L.orc_update.restype = C.c_long
        L.orc_update.argtypes = [C.c_size_t, dp, dp, C.c_double, dp]
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.orc_direction.argtypes = [C.POINTER(C.c_uint32), C.c_int, dp]
        L.orc_direction_by_eye.argtypes = [C.POINTER(C.c_uint32), C.c_int, dp]
        _lib = L
    return _lib


def philox4x32_10(key, ctr):
    k = (C.c_uint32 * 2)(*key)
    c = (C.c_uint32 * 4)(*ctr)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(k, c, o)
    return tuple(int(v) for v in o)


def direction(words, use_float=False):
    """O6 of the chain: the unit vector made from the four words of one Philox call."""
    x = (C.c_uint32 * 4)(*[int(w) for w in words])
    out = np.zeros(3)
    lib().orc_direction(x, int(use_float), _dp(out))
    return out


def direction_by_eye(words, use_float=False):
    """The same lattice point as direction(), from the definition of a unit vector with the C library's cosl / sinl
    (not used by the chain; the readable twin of O6)."""
    x = (C.c_uint32 * 4)(*[int(w) for w in words])
    out = np.zeros(3)
    lib().orc_direction_by_eye(x, int(use_float), _dp(out))
    return out


def threads() -> int:
    return int(lib().orc_threads())


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


TRACE_FIELDS = ("E1", "E2", "E3", "s", "t", "pf", "w", "f1", "f2", "f3", "f4", "gain", "loss", "u")


class Oracle:
    """Handle on one problem (species, grids, processes).  ``problem`` is the plain dict produced by
    ``workloads.configs`` (keys: nx, species, grids, processes, hbar)."""

    def __init__(self, problem: dict, use_float: bool = False):
        L = lib()
        sp = problem["species"]
        gr = problem["grids"]
        pr = problem["processes"]
        self.nx = int(problem["nx"])
        S = (_Species * len(sp))(*[_Species(s["mass"], s.get("charge", 0.0), s["stat"], s.get("g", 1.0)) for s in sp])
        G = (_Grid * len(gr))(*[_Grid((C.c_int * 3)(*g["n"]), (C.c_double * 3)(*g["pmin"]),
                                      (C.c_double * 3)(*g["pmax"])) for g in gr])
        P = (_Process * len(pr))(*[_Process(p["a"], p["b"], p["c"], p["d"], p["kind"],
                                            (C.c_double * 4)(*(list(p["par"]) + [0.0] * 4)[:4]),
                                            p.get("sym", -1.0), int(p.get("sampler", 0))) for p in pr])
        self._h = L.orc_create(self.nx, len(sp), S, G, len(pr), P, float(problem.get("hbar", 1.0)), int(use_float))
        if not self._h:
            raise ValueError("oracle: unsupported problem (unknown kind or sampler; a+b->b+a must be written a+b->a+b; sampler 1 needs "
                             "an elastic t-channel kind; a species in a process must have no cell centre with p0 = 0, Eq. 16's 1/p0)")
        self.n_species = len(sp)
        self.np = [int(np.prod(g["n"])) for g in gr]
        self.f_elems = int(L.orc_f_elems(self._h))
        self.detail_elems = int(L.orc_detail_elems(self._h))
        self.n_roles = int(L.orc_n_roles(self._h))
        self.sp_off = [int(L.orc_species_offset(self._h, s)) for s in range(len(sp))]
        self.role_off = [int(L.orc_role_offset(self._h, r)) for r in range(self.n_roles)]
        self.roles = []
        for r in range(self.n_roles):
            s4 = (C.c_int * 4)()
            kind, sym, proc = C.c_int(), C.c_double(), C.c_int()
            L.orc_role_info(self._h, r, s4, C.byref(kind), C.byref(sym), C.byref(proc))
            self.roles.append(dict(s=tuple(s4), kind=kind.value, sym=sym.value, process=proc.value))

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:      # at interpreter shutdown the module globals may be gone
            _lib.orc_destroy(self._h)
            self._h = None

    def _cb(self, fcb):
        """fcb: None (grid mode), a Python callable f(species, (px,py,pz)), or ('thermal', rows) with
        one row (scale, T, mu, m, theta, ux, uy, uz) per species for the built-in analytic family."""
        if fcb is None:
            return None, None
        if isinstance(fcb, tuple) and fcb[0] == "thermal":
            arr = np.ascontiguousarray(fcb[1], dtype=np.float64).reshape(self.n_species, 8)
            self._user_keep = arr
            return arr, (C.cast(lib().orc_builtin_thermal, C.c_void_p), arr.ctypes.data_as(C.c_void_p))
        def tramp(species, p, _user):
            return float(fcb(species, (p[0], p[1], p[2])))
        c = FCALLBACK(tramp)
        return c, (C.cast(c, C.c_void_p), None)

    @staticmethod
    def _fp(ptr):
        return (None, None) if ptr is None else ptr

    def collision(self, f, n_samples, seed, ix_begin=0, ix_end=None, ix_stride=1, detail=False, fcb=None,
                  box_cut=True):
        """Returns C (f_elems doubles; only visited spatial cells written, rest 0) and, with
        ``detail``, a dict of per-(role, ix, p1) arrays G, L, Lin, Q."""
        f = np.ascontiguousarray(f, dtype=np.float64) if f is not None else np.zeros(self.f_elems)
        assert f.size == self.f_elems
        Cout = np.zeros(self.f_elems)
        ix_end = self.nx if ix_end is None else ix_end
        d = {k: np.zeros(self.detail_elems) for k in ("G", "L", "Lin", "Q")} if detail else {}
        keep, ptr = self._cb(fcb)
        rc = lib().orc_collision(self._h, _dp(f), _dp(Cout), int(n_samples), int(seed), ix_begin, ix_end, ix_stride,
                                 _dp(d.get("G")), _dp(d.get("L")), _dp(d.get("Lin")), _dp(d.get("Q")), *self._fp(ptr),
                                 int(box_cut))
        if rc != 0:
            raise ValueError("oracle: bad arguments")
        return (Cout, d) if detail else Cout

    def collision_symmetric(self, f, n_samples, seed, ix_begin=0, ix_end=None, ix_stride=1, slot_mask=15):
        """NEXT-3: the conservative ("symmetric") estimator (rbg_oracle.cpp, SymSink).  Returns (C, mag): mag is the sum
        of the absolute deposits per cell, the scale of the parity tolerance.  slot_mask (tests): deposit only for the
        slots whose bit is set, to isolate one slot's estimator."""
        f = np.ascontiguousarray(f, dtype=np.float64)
        assert f.size == self.f_elems
        Cout, mag = np.zeros(self.f_elems), np.zeros(self.f_elems)
        ix_end = self.nx if ix_end is None else ix_end
        rc = lib().orc_collision_symmetric(self._h, _dp(f), _dp(Cout), _dp(mag), int(n_samples), int(seed), ix_begin, ix_end,
                                           ix_stride, int(slot_mask))
        if rc != 0:
            raise ValueError("oracle: bad arguments")
        return Cout, mag

    def point(self, f, role, ix, ip1, n_samples, seed, fcb=None, box_cut=True):
        """Scaled (G, L, Lin, Q) of one (role, ix, p1); C_role = G - L, stderr = sqrt(Q - (G-L)^2/N)."""
        f = np.ascontiguousarray(f, dtype=np.float64) if f is not None else np.zeros(self.f_elems)
        out = np.zeros(4)
        keep, ptr = self._cb(fcb)
        lib().orc_collision_point(self._h, _dp(f), role, ix, ip1, int(n_samples), int(seed), _dp(out), *self._fp(ptr),
                                  int(box_cut))
        return out

    def m2_qcd(self, role, s, t, u):
        """|M|^2(s,t,u) of a Table III role as the sample loop evaluates it."""
        return float(lib().orc_m2_qcd(self._h, int(role), float(s), float(t), float(u)))

    def trace(self, f, role, ix, ip1, n, seed, fcb=None, box_cut=True):
        f = np.ascontiguousarray(f, dtype=np.float64) if f is not None else np.zeros(self.f_elems)
        dout = np.zeros(26)
        iout = (C.c_int * 5)()
        keep, ptr = self._cb(fcb)
        lib().orc_trace(self._h, _dp(f), role, ix, ip1, n, int(seed), _dp(dout), iout, *self._fp(ptr), int(box_cut))
        t = dict(p1=dout[0:3].copy(), p2=dout[3:6].copy(), p3=dout[6:9].copy(), p4=dout[9:12].copy())
        t.update({k: float(dout[12 + i]) for i, k in enumerate(TRACE_FIELDS)})
        t.update(j2=iout[0], j3=iout[1], j4=iout[2], status=iout[3], draws=iout[4])
        return t


def update(f, Cterm, dt):
    """Eq. 27 explicit Euler: f_out = f + dt*C and the count of negative cells."""
    f = np.ascontiguousarray(f, dtype=np.float64)
    Cterm = np.ascontiguousarray(Cterm, dtype=np.float64)
    out = np.empty_like(f)
    neg = lib().orc_update(f.size, _dp(f), _dp(Cterm), float(dt), _dp(out))
    return out, int(neg)
