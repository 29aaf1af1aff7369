"""ctypes marshalling for librbg.so; names follow include/rbg.h one to one."""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

KIND_CONST, KIND_COULOMB_SCREENED, KIND_TCHAN_S2, KIND_ISO_DSIGMA = 0, 1, 2, 3
# Table III
(KIND_QCD_Q1Q2, KIND_QCD_Q1Q1, KIND_QCD_Q1QB1, KIND_QCD_Q1QB1_Q2QB2, KIND_QCD_QQB_GG, KIND_QCD_QG,
 KIND_QCD_GG) = 4, 5, 6, 7, 8, 9, 10
RBG_FP64, RBG_FP32_KINEMATICS = 0, 1
SAMPLER_UNIFORM, SAMPLER_TCHANNEL = 0, 1

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "librbg.so"
_lib = None


class RbgError(RuntimeError):
    pass


class _SpatialGrid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ix_offset", C.c_int)]


class _MomentumGrid(C.Structure):
    _fields_ = [("n", C.c_int * 3), ("pmin", C.c_double * 3), ("pmax", C.c_double * 3)]


class _Species(C.Structure):
    _fields_ = [("mass", C.c_double), ("charge", C.c_double), ("stat", C.c_int), ("g", C.c_double)]


class _DriftParams(C.Structure):
    _fields_ = [("dt", C.c_double), ("dx", C.c_double * 3), ("bc", C.c_int * 3), ("zeta", C.c_double)]


class _BeStepParams(C.Structure):
    _fields_ = [("dt", C.c_double), ("dx", C.c_double * 3), ("bc", C.c_int * 3), ("zeta", C.c_double),
                ("n_samples", C.c_int), ("seed", C.c_uint64), ("do_drift", C.c_int), ("do_vlasov", C.c_int),
                ("do_collision", C.c_int)]


N_MOMENTS = 14


class _Process(C.Structure):
    _fields_ = [("a", C.c_int), ("b", C.c_int), ("c", C.c_int), ("d", C.c_int), ("kind", C.c_int),
                ("par", C.c_double * 4), ("sym", C.c_double), ("sampler", C.c_int)]


# every symbol include/rbg.h declares
_SIGNATURES = {
    "rbg_create": (C.c_int, [C.POINTER(C.c_void_p), C.POINTER(_SpatialGrid), C.c_int, C.POINTER(_Species),
                             C.POINTER(_MomentumGrid), C.c_int, C.POINTER(_Process), C.c_double, C.c_int]),
    "rbg_collision": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_uint64, C.c_void_p]),
    "rbg_collision_symmetric": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_uint64, C.c_void_p]),
    "rbg_collision_update": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_int,
                                       C.c_uint64, C.c_void_p]),
    "rbg_collision_evolve": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_int, C.c_void_p, C.c_int,
                                       C.c_uint64, C.c_void_p]),
    "rbg_collision_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_uint64]),
    "rbg_collision_update_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.POINTER(C.c_int), C.c_int, C.c_uint64]),
    "rbg_moments": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "rbg_moments_static": (C.c_int, [C.POINTER(_MomentumGrid), C.c_double, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]),
    "rbg_drift_step": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "rbg_drift_step_pfl": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.POINTER(C.c_double), C.c_void_p]),
    "rbg_vlasov_step": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]),
    "rbg_be_step": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "rbg_f_elems": (C.c_size_t, [C.c_void_p]),
    "rbg_n_roles": (C.c_int, [C.c_void_p]),
    "rbg_role_info": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_double), C.POINTER(C.c_double),
                                C.POINTER(C.c_double), C.POINTER(C.c_int)]),
    "rbg_sample_evals": (C.c_uint64, [C.c_void_p, C.c_int]),
    "rbg_last_launch_count": (C.c_int, [C.c_void_p]),
    "rbg_set_option": (C.c_int, [C.c_void_p, C.c_char_p, C.c_int]),
    "rbg_last_error": (C.c_char_p, [C.c_void_p]),
    "rbg_destroy": (None, [C.c_void_p]),
    "rbg_probe_alu_peak": (C.c_int, [C.c_int, C.c_int, C.POINTER(C.c_double), C.c_void_p]),
    "rbg_selftest_math": (C.c_int, [C.c_uint64, C.c_uint32, C.POINTER(C.c_uint64)]),
    "rbg_selfcheck_failures": (C.c_int, [C.POINTER(C.c_uint64)]),
}


def exported_symbols():
    return sorted(_SIGNATURES)


def use_checked_build():
    """Select librbg_checked.so (device-side index / layout / ring-slot checks, rbg_selfcheck_failures) for this process.
    Must be called before the first load_library()."""
    global _LIB_PATH
    if _lib is not None:
        raise RbgError("the library is already loaded")
    _LIB_PATH = _PKG / "librbg_checked.so"


def load_library():
    """Load librbg.so; raises RbgError if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not _LIB_PATH.exists():
            raise RbgError(f"{_LIB_PATH} is missing: run `python -m paper_2308_04869_b200.build` "
                           "(there is no CPU fallback)")
        lib = C.CDLL(str(_LIB_PATH))
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def _check(rc, handle=None):
    if rc != 0:
        msg = load_library().rbg_last_error(handle)
        raise RbgError(f"librbg error {rc}: {msg.decode() if msg else ''}")


def probe_alu_peak(what: int, iters: int = 1 << 16, stream=None) -> float:
    """Operations/s (one FMA or multiply = one op) of a register-resident chain: 0 fp64, 1 fp32, 2 int32 (two of three
    operands re-used), 3 fp64 with three distinct register operands per FMA, 4 the 32 x 32 -> 64-bit multiply of Philox."""
    out = C.c_double()
    _check(load_library().rbg_probe_alu_peak(what, iters, C.byref(out), _stream_ptr(stream)))
    return out.value


def selfcheck_failures():
    """rbg_selfcheck_failures: the eight failure counters of the checked build (raises in the normal build)."""
    out = (C.c_uint64 * 8)()
    _check(load_library().rbg_selfcheck_failures(out))
    return [int(v) for v in out]


def selftest_math(n_operands: int, seed: int = 1) -> int:
    """rbg_selftest_math: number of bitwise mismatches (must be 0)."""
    out = C.c_uint64()
    _check(load_library().rbg_selftest_math(int(n_operands), int(seed), C.byref(out)))
    return int(out.value)


def _stream_ptr(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(getattr(stream, "cuda_stream", stream))


MOMENTS_STATIC_MAX_CELLS = 65536


def moments_static(grid: dict, mass: float, f, out=None, stream=None):
    """rbg_moments_static: the 14 moments of one species, M[n_cells, 14], with no handle and no device allocation inside
    the library -- for programs that cannot let a library call cudaMalloc where they need the moments (all of HBM already
    in their own pool, a time-step loop that must not hit cudaMalloc's device-wide synchronisation, a host application
    that forbids allocations after start-up).  The species' 1/E_p table sits in a fixed 512 KB array inside librbg.so, so
    the momentum grid may have at most MOMENTS_STATIC_MAX_CELLS cells (larger: RbgError, nothing is truncated).

    ``grid`` = dict(n, pmin, pmax); ``f`` = that species' block, a contiguous float64 CUDA tensor of n_cells * prod(n)
    elements on the current device.  Pass ``out`` (float64 CUDA, n_cells * 14 elements) to keep this wrapper from allocating
    as well; without it the result tensor comes from torch's allocator.  The first call on a device looks up the array's
    address: make it before any stream capture.  Calls share the array, so keep them on one stream (include/rbg.h)."""
    import torch
    npc = int(np.prod(grid["n"]))
    if not (isinstance(f, torch.Tensor) and f.is_cuda and f.dtype == torch.float64 and f.is_contiguous()
            and npc > 0 and f.numel() % npc == 0):
        raise RbgError("f must be a contiguous float64 CUDA tensor holding whole spatial cells of this momentum grid")
    n_cells = f.numel() // npc
    if out is None:
        out = torch.empty((n_cells, N_MOMENTS), dtype=torch.float64, device=f.device)
    elif not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.is_contiguous()
              and out.numel() == n_cells * N_MOMENTS and out.device == f.device):
        raise RbgError(f"out must be a contiguous float64 CUDA tensor with {n_cells * N_MOMENTS} elements on f's device")
    g = _MomentumGrid((C.c_int * 3)(*grid["n"]), (C.c_double * 3)(*grid["pmin"]), (C.c_double * 3)(*grid["pmax"]))
    _check(load_library().rbg_moments_static(C.byref(g), float(mass), int(n_cells), C.c_void_p(f.data_ptr()),
                                             C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
    return out


class Collision:
    """One problem (spatial cells, species, momentum grids, processes) on the current CUDA device.

    ``problem`` is a plain dict: nx (number of spatial cells, or (nx,ny,nz)), species [dict(mass,
    charge, stat, g)], grids [dict(n, pmin, pmax)], processes [dict(a,b,c,d,kind,par,sym)], hbar.
    """

    def __init__(self, problem: dict, fp32_kinematics: bool = False, ix_offset: int = 0):
        lib = load_library()
        nx = problem["nx"]
        nxyz = (int(nx), 1, 1) if np.isscalar(nx) else tuple(int(v) for v in nx)
        sg = _SpatialGrid(*nxyz, int(ix_offset))
        sp, gr, pr = problem["species"], problem["grids"], problem["processes"]
        S = (_Species * len(sp))(*[_Species(s["mass"], s.get("charge", 0.0), s["stat"], s.get("g", 1.0)) for s in sp])
        G = (_MomentumGrid * len(gr))(*[_MomentumGrid((C.c_int * 3)(*g["n"]), (C.c_double * 3)(*g["pmin"]),
                                                      (C.c_double * 3)(*g["pmax"])) for g in gr])
        P = (_Process * max(len(pr), 1))(*[_Process(p["a"], p["b"], p["c"], p["d"], p["kind"],
                                                    (C.c_double * 4)(*(list(p["par"]) + [0.0] * 4)[:4]),
                                                    p.get("sym", -1.0), int(p.get("sampler", 0))) for p in pr])
        h = C.c_void_p()
        _check(lib.rbg_create(C.byref(h), C.byref(sg), len(sp), S, G, len(pr), P, float(problem.get("hbar", 1.0)),
                              RBG_FP32_KINEMATICS if fp32_kinematics else RBG_FP64))
        self._h = h
        self.f_elems = int(lib.rbg_f_elems(h))
        self.n_roles = int(lib.rbg_n_roles(h))
        self.n_species = len(sp)
        self.n_cells = int(np.prod(nxyz))

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            load_library().rbg_destroy(h)
            self._h = None

    # -- helpers ---------------------------------------------------------------------------------
    def _dev(self, t, name):
        import torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and t.numel() == self.f_elems):
            raise RbgError(f"{name} must be a contiguous float64 CUDA tensor with {self.f_elems} elements")
        return C.c_void_p(t.data_ptr())

    def sample_evals(self, n_samples: int) -> int:
        return int(load_library().rbg_sample_evals(self._h, int(n_samples)))

    def role_info(self, r: int) -> dict:
        """rbg_role_info: dict(s=(s1, s2, s3, s4), sym, cl, cg, process) of role r as the library expanded it."""
        s4 = (C.c_int * 4)()
        sym, cl, cg, proc = C.c_double(), C.c_double(), C.c_double(), C.c_int()
        _check(load_library().rbg_role_info(self._h, int(r), s4, C.byref(sym), C.byref(cl), C.byref(cg), C.byref(proc)), self._h)
        return dict(s=tuple(s4), sym=sym.value, cl=cl.value, cg=cg.value, process=proc.value)

    def last_launch_count(self) -> int:
        return int(load_library().rbg_last_launch_count(self._h))

    def set_option(self, key: str, value: int):
        _check(load_library().rbg_set_option(self._h, key.encode(), int(value)), self._h)

    # -- the hot path ----------------------------------------------------------------------------
    def collision(self, f, n_samples: int, seed: int, out=None, stream=None):
        """rbg_collision: C[f] for every cell (torch CUDA tensors; asynchronous on the stream)."""
        import torch
        if out is None:
            out = torch.empty_like(f)
        _check(load_library().rbg_collision(self._h, self._dev(f, "f"), self._dev(out, "out"), int(n_samples),
                                            int(seed), _stream_ptr(stream)), self._h)
        return out

    def collision_symmetric(self, f, n_samples: int, seed: int, out=None, stream=None):
        """rbg_collision_symmetric: the conservative ("symmetric") estimator of C[f] (NEXT-3)."""
        import torch
        if out is None:
            out = torch.empty_like(f)
        _check(load_library().rbg_collision_symmetric(self._h, self._dev(f, "f"), self._dev(out, "out"), int(n_samples),
                                                      int(seed), _stream_ptr(stream)), self._h)
        return out

    def collision_update(self, f, dt: float, n_samples: int, seed: int, out=None, neg_flag=None, stream=None):
        """rbg_collision_update: f_out = f + dt*C[f]; neg_flag (int32 CUDA tensor) += #cells with f_out < 0."""
        import torch
        if out is None:
            out = torch.empty_like(f)
        if neg_flag is None:
            neg_flag = torch.zeros(1, dtype=torch.int32, device=f.device)
        _check(load_library().rbg_collision_update(self._h, self._dev(f, "f"), self._dev(out, "out"), float(dt),
                                                   C.c_void_p(neg_flag.data_ptr()), int(n_samples), int(seed),
                                                   _stream_ptr(stream)), self._h)
        return out, neg_flag

    def collision_evolve(self, f, dt: float, n_steps: int, n_samples: int, seed: int, scratch=None, neg_flag=None,
                         stream=None):
        """rbg_collision_evolve: n_steps Euler steps f <- f + dt*C[f] in place (step k uses seed + k)."""
        import torch
        if scratch is None:
            scratch = torch.empty_like(f)
        if neg_flag is None:
            neg_flag = torch.zeros(1, dtype=torch.int32, device=f.device)
        _check(load_library().rbg_collision_evolve(self._h, self._dev(f, "f"), self._dev(scratch, "scratch"), float(dt),
                                                   int(n_steps), C.c_void_p(neg_flag.data_ptr()), int(n_samples),
                                                   int(seed), _stream_ptr(stream)), self._h)
        return f, neg_flag

    # -- the steps either side of the collision term (NEXT-4) --------------------------------------
    def moments(self, f, stream=None):
        """rbg_moments: (M[n_species, Nx, 14], total[Nx, 14], em[Nx, 4]) as CUDA tensors."""
        import torch
        M = torch.empty((self.n_species, self.n_cells, N_MOMENTS), dtype=torch.float64, device=f.device)
        tot = torch.empty((self.n_cells, N_MOMENTS), dtype=torch.float64, device=f.device)
        em = torch.empty((self.n_cells, 4), dtype=torch.float64, device=f.device)
        _check(load_library().rbg_moments(self._h, self._dev(f, "f"), C.c_void_p(M.data_ptr()), C.c_void_p(tot.data_ptr()),
                                          C.c_void_p(em.data_ptr()), _stream_ptr(stream)), self._h)
        return M, tot, em

    def drift_step(self, f, dt: float, dx, bc=(1, 1, 1), zeta: float = 0.0, out=None, stream=None):
        """rbg_drift_step: one UPFD step of the drift term (Eq. 30)."""
        import torch
        if out is None:
            out = torch.empty_like(f)
        p = _DriftParams(float(dt), (C.c_double * 3)(*[float(v) for v in dx]), (C.c_int * 3)(*[int(v) for v in bc]), float(zeta))
        _check(load_library().rbg_drift_step(self._h, self._dev(f, "f"), self._dev(out, "out"), C.byref(p),
                                             _stream_ptr(stream)), self._h)
        return out

    def drift_step_pfl(self, f, dt: float, dx, out=None, stream=None):
        """rbg_drift_step_pfl: one step of the second-order flux-limited drift scheme (Eq. 31-33), periodic."""
        import torch
        if out is None:
            out = torch.empty_like(f)
        _check(load_library().rbg_drift_step_pfl(self._h, self._dev(f, "f"), self._dev(out, "out"), float(dt),
                                                 (C.c_double * 3)(*[float(v) for v in dx]), _stream_ptr(stream)), self._h)
        return out

    def vlasov_step(self, f, dt: float, E, B, out=None, stream=None):
        """rbg_vlasov_step: one UPFD step of the Vlasov term (Eq. 34); E, B are [Nx, 3] float64 CUDA tensors."""
        import torch
        if out is None:
            out = torch.empty_like(f)
        for name, t in (("E", E), ("B", B)):
            if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                    and t.numel() == 3 * self.n_cells):
                raise RbgError(f"{name} must be a contiguous float64 CUDA tensor with {3 * self.n_cells} elements")
        _check(load_library().rbg_vlasov_step(self._h, self._dev(f, "f"), self._dev(out, "out"), float(dt),
                                              C.c_void_p(E.data_ptr()), C.c_void_p(B.data_ptr()), _stream_ptr(stream)),
               self._h)
        return out

    def be_step(self, f, dt: float, dx=(1.0, 1.0, 1.0), bc=(1, 1, 1), zeta: float = 0.0, E=None, B=None, n_samples: int = 0,
                seed: int = 0, drift=True, vlasov=True, collision=True, scratch=None, neg_flag=None, stream=None):
        """rbg_be_step: one time step of Eq. 25-27 in place (drift, Vlasov, collision with 3 dt).  collision="symmetric"
        uses the conservative estimator for the collision sub-step."""
        import torch
        if scratch is None:
            scratch = torch.empty_like(f)
        if neg_flag is None:
            neg_flag = torch.zeros(1, dtype=torch.int32, device=f.device)
        p = _BeStepParams(float(dt), (C.c_double * 3)(*[float(v) for v in dx]), (C.c_int * 3)(*[int(v) for v in bc]),
                          float(zeta), int(n_samples), int(seed), int(bool(drift)), int(bool(vlasov)), 2 if collision == "symmetric" else int(bool(collision)))
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        _check(load_library().rbg_be_step(self._h, self._dev(f, "f"), self._dev(scratch, "scratch"), C.byref(p), ptr(E), ptr(B),
                                          C.c_void_p(neg_flag.data_ptr()), _stream_ptr(stream)), self._h)
        return f, neg_flag

    def collision_update_host(self, f_host, dt: float, n_samples: int, seed: int, out=None):
        """rbg_collision_update_host: (f + dt*C[f], number of negative cells), host buffers in and out."""
        return self._host_call(f_host, n_samples, seed, out, dt)

    def collision_host(self, f_host, n_samples: int, seed: int, out=None):
        """rbg_collision_host: host buffers in, host buffers out (numpy float64 or pinned CPU tensors)."""
        return self._host_call(f_host, n_samples, seed, out, None)

    def _host_call(self, f_host, n_samples, seed, out, dt):
        import torch
        def ptr(a, name):
            if isinstance(a, torch.Tensor):
                ok = (not a.is_cuda) and a.dtype == torch.float64 and a.is_contiguous() and a.numel() == self.f_elems
                p = a.data_ptr()
            else:
                ok = a.dtype == np.float64 and a.flags.c_contiguous and a.size == self.f_elems
                p = a.ctypes.data
            if not ok:
                raise RbgError(f"{name} must be a contiguous float64 host array with {self.f_elems} elements")
            return C.c_void_p(p)
        if out is None:
            out = torch.empty_like(f_host) if isinstance(f_host, torch.Tensor) else np.empty_like(f_host)
        if dt is not None:
            neg = C.c_int(0)
            _check(load_library().rbg_collision_update_host(self._h, ptr(f_host, "f_host"), ptr(out, "out"), float(dt),
                                                            C.byref(neg), int(n_samples), int(seed)), self._h)
            return out, int(neg.value)
        _check(load_library().rbg_collision_host(self._h, ptr(f_host, "f_host"), ptr(out, "out"), int(n_samples),
                                                 int(seed)), self._h)
        return out
