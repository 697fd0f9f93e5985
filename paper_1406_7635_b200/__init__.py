"""Thin Python binding of libmm_b200.so (C ABI in include/mm.h).

Argument marshalling only: every step of the path runs in the CUDA kernels of csrc/.  PyTorch is
used for device memory (its caching allocator backs the handle through mm_create_ex) and for the
CUDA stream.  There is no CPU fallback: without the built library, or without a CUDA device,
calls raise.  Function names follow the C ABI; `Sim` is a convenience wrapper over them.
"""
import ctypes as C
import os

import numpy as np

MM_OK, MM_EINVAL, MM_ENOMEM, MM_ECUDA, MM_ESTATE, MM_ENAN, MM_EDT = 0, -1, -2, -3, -4, -5, -6
MM_DEMAG, MM_EXCH, MM_ANIS, MM_ZEEMAN, MM_ALL = 1, 2, 4, 8, 15
MM_MAX_REGIONS = 256
MM_OPT_GENERIC_FFT = 1
MM_OPT_NO_TMA = 2
MM_OPT_NO_GRAPH = 3
MM_RK45, MM_RK23, MM_RK12 = 0, 1, 2

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("MM_B200_LIB") or os.path.join(_HERE, "libmm_b200.so")     # (the variable: another build of the same library)
_lib_handle = None


class MMError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("mm error %d: %s" % (code, text))
        self.code = code


class mm_params(C.Structure):
    _fields_ = [
        ("nregions", C.c_int),
        ("Msat", C.c_double * MM_MAX_REGIONS), ("Aex", C.c_double * MM_MAX_REGIONS),
        ("alpha", C.c_double * MM_MAX_REGIONS),
        ("Ku1", C.c_double * MM_MAX_REGIONS), ("Ku2", C.c_double * MM_MAX_REGIONS),
        ("anisU", (C.c_double * 3) * MM_MAX_REGIONS),
        ("Kc1", C.c_double * MM_MAX_REGIONS), ("Kc2", C.c_double * MM_MAX_REGIONS),
        ("Kc3", C.c_double * MM_MAX_REGIONS),
        ("anisC1", (C.c_double * 3) * MM_MAX_REGIONS), ("anisC2", (C.c_double * 3) * MM_MAX_REGIONS),
        ("B_ext", C.c_double * 3),
        ("exch_scale", C.POINTER(C.c_double)),
        ("gamma_LL", C.c_double),
    ]


class mm_step_info(C.Structure):
    _fields_ = [("t", C.c_double), ("dt_taken", C.c_double), ("dt_next", C.c_double), ("err", C.c_double),
                ("accepted", C.c_int), ("n_eval", C.c_long)]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)

_SIGNATURES = {
    "mm_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                            C.c_int, C.c_int, C.c_int]),
    "mm_create_ex": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                               C.c_int, C.c_int, C.c_int, ALLOC_FN, FREE_FN, C.c_void_p, C.c_void_p]),
    "mm_destroy": (C.c_int, [C.c_void_p]),
    "mm_set_regions": (C.c_int, [C.c_void_p, C.c_void_p]),
    "mm_set_geometry": (C.c_int, [C.c_void_p, C.c_void_p]),
    "mm_set_params": (C.c_int, [C.c_void_p, C.POINTER(mm_params)]),
    "mm_set_terms": (C.c_int, [C.c_void_p, C.c_uint]),
    "mm_set_option": (C.c_int, [C.c_void_p, C.c_int, C.c_int]),
    "mm_set_solver": (C.c_int, [C.c_void_p] + [C.c_double] * 6),
    "mm_set_m": (C.c_int, [C.c_void_p, C.c_void_p]),
    "mm_get_m": (C.c_int, [C.c_void_p, C.c_void_p]),
    "mm_b_eff": (C.c_int, [C.c_void_p, C.c_uint, C.c_void_p]),
    "mm_torque": (C.c_int, [C.c_void_p, C.c_void_p]),
    "mm_set_solver_kind": (C.c_int, [C.c_void_p, C.c_int]),
    "mm_set_precession": (C.c_int, [C.c_void_p, C.c_int]),
    "mm_set_dmi": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.c_int]),
    "mm_set_zhang_li": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.c_double]),
    "mm_set_slonczewski": (C.c_int, [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double)]),
    "mm_set_temperature": (C.c_int, [C.c_void_p, C.c_double, C.c_ulonglong]),
    "mm_step_rk45": (C.c_int, [C.c_void_p, C.POINTER(mm_step_info)]),
    "mm_step": (C.c_int, [C.c_void_p, C.POINTER(mm_step_info)]),
    "mm_steps": (C.c_int, [C.c_void_p, C.c_int]),
    "mm_run": (C.c_int, [C.c_void_p, C.c_double]),
    "mm_energy": (C.c_int, [C.c_void_p, C.c_uint, C.POINTER(C.c_double)]),
    "mm_max_torque": (C.c_int, [C.c_void_p, C.POINTER(C.c_double)]),
    "mm_relax": (C.c_int, [C.c_void_p]),
    "mm_batch_steps": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int]),
    "mm_batch_run": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_double]),
    "mm_batch_relax": (C.c_int, [C.POINTER(C.c_void_p), C.c_int]),
    "mm_get_time": (C.c_int, [C.c_void_p, C.POINTER(C.c_double)]),
    "mm_set_time": (C.c_int, [C.c_void_p, C.c_double]),
    "mm_get_avg_m": (C.c_int, [C.c_void_p, C.POINTER(C.c_double)]),
    "mm_avg_m_noalloc": (C.c_int, [C.c_void_p, C.c_longlong, C.c_void_p, C.c_void_p, C.c_char_p, C.c_size_t]),
    "mm_get_stats": (C.c_int, [C.c_void_p, C.POINTER(C.c_long), C.POINTER(C.c_long), C.POINTER(C.c_long),
                               C.POINTER(C.c_size_t)]),
    "mm_get_memory": (C.c_int, [C.c_void_p, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]),
    "mm_get_stream": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p)]),
    "mm_get_fft_size": (C.c_int, [C.c_void_p, C.POINTER(C.c_int)]),
    "mm_get_launch_count": (C.c_int, [C.c_void_p, C.POINTER(C.c_long)]),
    "mm_profile": (C.c_int, [C.c_void_p, C.c_int]),
    "mm_profile_read": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_double),
                                  C.POINTER(C.c_long)]),
    "mm_last_error": (C.c_char_p, [C.c_void_p]),
    "mm_strerror": (C.c_char_p, [C.c_int]),
    "mm_version": (C.c_char_p, []),
}
EXPORTS = tuple(_SIGNATURES)


def lib():
    """Load libmm_b200.so (built in-tree by build.py / __graft_entry__.build()); raises if missing."""
    global _lib_handle
    if _lib_handle is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libmm_b200.so is not built (run `python -m paper_1406_7635_b200.build`); "
                               "there is no CPU fallback")
        h = C.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(h, name)
            fn.restype, fn.argtypes = res, args
        _lib_handle = h
    return _lib_handle


def _check(code, handle=None):
    if code != MM_OK:
        text = lib().mm_strerror(code).decode()
        if handle:
            detail = lib().mm_last_error(handle).decode()
            if detail:
                text += " (" + detail + ")"
        raise MMError(code, text)


def _ptr(a):
    """Raw pointer of a numpy array (host) or a torch tensor (host or device); keeps nothing alive."""
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return C.c_void_p(a.ctypes.data)
    assert a.is_contiguous()
    return C.c_void_p(a.data_ptr())


def make_params(p):
    """synth.Params (or any object with the same attributes) -> mm_params; returns (struct, keepalive)."""
    n = int(p.nregions)
    s = mm_params()
    s.nregions = n
    for name in ("Msat", "Aex", "alpha", "Ku1", "Ku2", "Kc1", "Kc2", "Kc3"):
        arr = np.asarray(getattr(p, name), dtype=np.float64)
        getattr(s, name)[:n] = arr[:n].tolist()
    for name in ("anisU", "anisC1", "anisC2"):
        arr = np.asarray(getattr(p, name), dtype=np.float64)
        dst = getattr(s, name)
        for r in range(n):
            dst[r][:] = arr[r].tolist()
    s.B_ext[:] = np.asarray(p.B_ext, dtype=np.float64).tolist()
    keep = None
    if p.exch_scale is not None:
        keep = np.ascontiguousarray(p.exch_scale, dtype=np.float64)
        s.exch_scale = keep.ctypes.data_as(C.POINTER(C.c_double))
    s.gamma_LL = float(p.gamma_LL)
    return s, keep


class Sim:
    """One simulation box on the current CUDA device; methods map 1:1 onto the mm_* calls."""

    def __init__(self, grid, cell, pbc=(0, 0, 0), use_torch_allocator=True, guard_bytes=0):
        """guard_bytes > 0 (debugging aid, with the torch allocator): every device buffer of the handle gets a guard
        zone of that many bytes on either side, filled with 0xA5; check_guards() tells whether any kernel wrote there."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the mm_b200 path has no CPU fallback")
        self._torch = torch
        self.grid = tuple(int(g) for g in grid)
        nx, ny, nz = self.grid
        self.ncells = nx * ny * nz
        self.shape = (3, nz, ny, nx)
        self._h = C.c_void_p()
        dev = torch.cuda.current_device()
        stream = torch.cuda.current_stream().cuda_stream     # 0 (the legacy default stream): the handle makes its own
        self._guards = {}
        if use_torch_allocator and guard_bytes:
            gb = (int(guard_bytes) + 255) // 256 * 256

            def _alloc(nbytes, ctx):
                try:
                    buf = torch.full((int(nbytes) + 2 * gb,), 0xA5, dtype=torch.uint8, device="cuda")
                except Exception:
                    return None
                self._guards[buf.data_ptr() + gb] = (buf, int(nbytes), gb)
                return buf.data_ptr() + gb

            def _free(ptr, ctx):
                self._guards.pop(ptr, None)
        elif use_torch_allocator:
            _new, _delete = torch.cuda.caching_allocator_alloc, torch.cuda.caching_allocator_delete

            def _alloc(nbytes, ctx):
                try:
                    return _new(int(nbytes), dev, stream)
                except Exception:
                    return None

            def _free(ptr, ctx):
                try:
                    _delete(ptr)
                except Exception:      # interpreter shutdown: torch is already gone
                    pass

        if use_torch_allocator:
            self._cb = (ALLOC_FN(_alloc), FREE_FN(_free))
            code = lib().mm_create_ex(C.byref(self._h), nx, ny, nz, cell[0], cell[1], cell[2], pbc[0], pbc[1], pbc[2],
                                      self._cb[0], self._cb[1], None, C.c_void_p(stream))
        else:
            code = lib().mm_create(C.byref(self._h), nx, ny, nz, cell[0], cell[1], cell[2], pbc[0], pbc[1], pbc[2])
        if code != MM_OK:
            raise MMError(code, lib().mm_strerror(code).decode() + " (" + lib().mm_last_error(None).decode() + ")")

    def check_guards(self):
        """Number of device buffers whose guard zones were written to (needs guard_bytes > 0 at construction)."""
        self._torch.cuda.synchronize()
        bad = 0
        for buf, n, gb in self._guards.values():
            if not (bool((buf[:gb] == 0xA5).all()) and bool((buf[gb + n:] == 0xA5).all())):
                bad += 1
        return bad

    @property
    def stream(self):
        """torch view of the CUDA stream the handle enqueues its work on (for events around its kernels)."""
        v = C.c_void_p()
        _check(lib().mm_get_stream(self._h, C.byref(v)), self._h)
        return self._torch.cuda.ExternalStream(v.value or 0)

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().mm_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- setters
    def set_regions(self, regions):
        if isinstance(regions, np.ndarray):
            regions = np.ascontiguousarray(regions, dtype=np.uint8)
        _check(lib().mm_set_regions(self._h, _ptr(regions)), self._h)

    def set_geometry(self, inside):
        """Shape of the magnet: one byte per cell [z][y][x], non-zero = inside (None removes it)."""
        if inside is None:
            _check(lib().mm_set_geometry(self._h, None), self._h)
            return
        if isinstance(inside, np.ndarray):
            inside = np.ascontiguousarray(inside, dtype=np.uint8)
        _check(lib().mm_set_geometry(self._h, _ptr(inside)), self._h)

    def set_params(self, p):
        s, keep = make_params(p)
        _check(lib().mm_set_params(self._h, C.byref(s)), self._h)

    def set_terms(self, mask):
        _check(lib().mm_set_terms(self._h, int(mask)), self._h)

    def set_option(self, option, value):
        _check(lib().mm_set_option(self._h, int(option), int(value)), self._h)

    def set_solver(self, max_err=0.0, headroom=0.0, fix_dt=0.0, dt_init=0.0, dt_min=0.0, dt_max=0.0):
        _check(lib().mm_set_solver(self._h, max_err, headroom, fix_dt, dt_init, dt_min, dt_max), self._h)

    def set_solver_kind(self, kind):
        """MM_RK45 (default) or MM_RK23."""
        _check(lib().mm_set_solver_kind(self._h, int(kind)), self._h)

    def set_temperature(self, kelvin, seed=0):
        _check(lib().mm_set_temperature(self._h, float(kelvin), int(seed)), self._h)

    def set_slonczewski(self, jz, pol, lam=1.0, eps_prime=0.0, mp=(0, 0, 1)):
        v = (C.c_double * 3)(*[float(x) for x in mp])
        _check(lib().mm_set_slonczewski(self._h, float(jz), float(pol), float(lam), float(eps_prime), v), self._h)

    def set_zhang_li(self, j, xi):
        v = (C.c_double * 3)(*[float(x) for x in j])
        _check(lib().mm_set_zhang_li(self._h, v, float(xi)), self._h)

    def set_dmi(self, D):
        """Dzyaloshinskii-Moriya strength [J/m^2]: a scalar or one value per region."""
        d = np.atleast_1d(np.asarray(D, dtype=np.float64))
        v = (C.c_double * len(d))(*d.tolist())
        _check(lib().mm_set_dmi(self._h, v, len(d)), self._h)

    def set_precession(self, on):
        _check(lib().mm_set_precession(self._h, 1 if on else 0), self._h)

    def set_m(self, m):
        if isinstance(m, np.ndarray):
            m = np.ascontiguousarray(m, dtype=np.float32)
        _check(lib().mm_set_m(self._h, _ptr(m)), self._h)

    # ---- getters (numpy by default; pass a torch CUDA tensor as `out` to stay on the device)
    def _out(self, out):
        return np.empty(self.shape, dtype=np.float32) if out is None else out

    def get_m(self, out=None):
        out = self._out(out)
        _check(lib().mm_get_m(self._h, _ptr(out)), self._h)
        return out

    def b_eff(self, term_mask=MM_ALL, out=None):
        out = self._out(out)
        _check(lib().mm_b_eff(self._h, int(term_mask), _ptr(out)), self._h)
        return out

    def torque(self, out=None):
        out = self._out(out)
        _check(lib().mm_torque(self._h, _ptr(out)), self._h)
        return out

    # ---- time stepping
    def step(self, want_info=True):
        if not want_info:
            _check(lib().mm_step_rk45(self._h, None), self._h)
            return None
        info = mm_step_info()
        _check(lib().mm_step_rk45(self._h, C.byref(info)), self._h)
        return dict(t=info.t, dt_taken=info.dt_taken, dt_next=info.dt_next, err=info.err,
                    accepted=bool(info.accepted), n_eval=info.n_eval)

    def steps(self, n):
        _check(lib().mm_steps(self._h, int(n)), self._h)

    def run(self, duration):
        _check(lib().mm_run(self._h, float(duration)), self._h)

    @property
    def t(self):
        v = C.c_double()
        _check(lib().mm_get_time(self._h, C.byref(v)), self._h)
        return v.value

    def energy(self, term_mask=MM_ALL):
        v = C.c_double()
        _check(lib().mm_energy(self._h, int(term_mask), C.byref(v)), self._h)
        return v.value

    def max_torque(self):
        v = C.c_double()
        _check(lib().mm_max_torque(self._h, C.byref(v)), self._h)
        return v.value

    def relax(self):
        _check(lib().mm_relax(self._h), self._h)

    def set_time(self, t):
        _check(lib().mm_set_time(self._h, float(t)), self._h)

    def avg_m(self):
        v = (C.c_double * 3)()
        _check(lib().mm_get_avg_m(self._h, v), self._h)
        return np.array(v[:])

    def stats(self):
        a, b, c, d = C.c_long(), C.c_long(), C.c_long(), C.c_size_t()
        _check(lib().mm_get_stats(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(d)), self._h)
        return dict(steps=a.value, rejected=b.value, evals=c.value, peak_device_bytes=d.value)

    def memory(self):
        """(resident, peak) device bytes owned by the handle."""
        a, b = C.c_size_t(), C.c_size_t()
        _check(lib().mm_get_memory(self._h, C.byref(a), C.byref(b)), self._h)
        return a.value, b.value

    def fft_size(self):
        v = (C.c_int * 3)()
        _check(lib().mm_get_fft_size(self._h, v), self._h)
        return tuple(v[:])

    def profile(self, enable):
        _check(lib().mm_profile(self._h, 1 if enable else 0), self._h)

    def profile_read(self):
        """{kernel class: (total ms, launches)} accumulated since profile(True)."""
        out = {}
        for kind in range(64):
            name, ms, n = C.c_char_p(), C.c_double(), C.c_long()
            if lib().mm_profile_read(self._h, kind, C.byref(name), C.byref(ms), C.byref(n)) != MM_OK:
                break
            if n.value:
                out[name.value.decode()] = (ms.value, n.value)
        return out

    def launch_count(self):
        v = C.c_long()
        _check(lib().mm_get_launch_count(self._h, C.byref(v)), self._h)
        return v.value


def _handles(sims):
    arr = (C.c_void_p * len(sims))(*[s._h.value for s in sims])
    return arr, len(sims)


def batch_steps(sims, n):
    """n attempted steps of every Sim in `sims`, concurrently (mm_batch_steps)."""
    arr, cnt = _handles(sims)
    _check(lib().mm_batch_steps(arr, cnt, int(n)))


def batch_run(sims, duration):
    arr, cnt = _handles(sims)
    _check(lib().mm_batch_run(arr, cnt, float(duration)))


def batch_relax(sims):
    arr, cnt = _handles(sims)
    _check(lib().mm_batch_relax(arr, cnt))


MM_NOALLOC_MAX_CELLS = 1 << 26


def avg_m_noalloc(m_dev, avg_dev, stream=None):
    """mm_avg_m_noalloc: mean of the device field `m_dev` (torch CUDA tensor, 3N floats) into `avg_dev` (torch CUDA
    tensor, 3 doubles) on `stream` (a raw cudaStream_t or None); allocates nothing and does not synchronise."""
    err = C.create_string_buffer(256)
    code = lib().mm_avg_m_noalloc(_ptr(m_dev), m_dev.numel() // 3, _ptr(avg_dev), C.c_void_p(stream or 0), err, len(err))
    if code != MM_OK:
        raise MMError(code, lib().mm_strerror(code).decode() + " (" + err.value.decode() + ")")


def from_config(cfg, **kw):
    """Build a Sim from a synth.configs dictionary (grid, cell, pbc, regions, params, m0)."""
    sim = Sim(cfg["grid"], cfg["cell"], cfg["pbc"], **kw)
    sim.set_params(cfg["params"])           # tables first: the region map is validated against them
    if cfg.get("regions") is not None:
        sim.set_regions(cfg["regions"])
    sim.set_m(cfg["m0"])
    return sim
