"""paper_2606_09356_b200 -- thin Python binding of libsoma_b200.so (include/soma.h).

Argument marshalling only: every step of the SCMF Monte-Carlo step runs in the library's sm_100a
kernels.  PyTorch is used for device memory (the workspace tensor, device-side result tensors) and
for the CUDA stream.  There is no CPU fallback: a missing library or device raises.

The functions carry the C names (`soma_create`, `soma_load_state`, `soma_mc_steps`,
`soma_get_density`, `soma_get_positions`, `soma_destroy`); `Soma` is a small convenience wrapper
over them.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional, Sequence

import numpy as np

from . import _build

SOMA_OK, SOMA_EINVAL, SOMA_ENOMEM, SOMA_ECUDA, SOMA_ESTATE = 0, -1, -2, -3, -4
_ERR = {SOMA_EINVAL: "SOMA_EINVAL", SOMA_ENOMEM: "SOMA_ENOMEM", SOMA_ECUDA: "SOMA_ECUDA", SOMA_ESTATE: "SOMA_ESTATE"}

LIB_PATH: Path = _build.LIB_PATH

# every symbol include/soma.h declares (tests check the library exports exactly these)
EXPORTS = (
    "soma_workspace_bytes", "soma_create", "soma_load_state", "soma_mc_steps", "soma_get_density",
    "soma_get_positions", "soma_get_omega", "soma_set_external_field", "soma_generate_state", "soma_init_from_density", "soma_validate_state", "soma_validate_noalloc", "soma_get_step", "soma_destroy", "soma_last_error",
    "soma_set_option", "soma_get_counters", "soma_get_kernel_times", "soma_debug_half_sweep", "soma_debug_finish_step",
    "soma_debug_set_omega", "soma_debug_philox", "soma_debug_maps", "soma_debug_accept",
    "soma_debug_accept_fma", "soma_debug_cell_index", "soma_debug_red_throughput",
)


class SomaError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"{_ERR.get(code, code)}: {text}")
        self.code = code


class soma_params(C.Structure):
    """Mirror of `struct soma_params` in include/soma.h."""
    _fields_ = [
        ("n_chains", C.c_uint64),
        ("beads_per_chain", C.c_uint32),
        ("n_types", C.c_uint32),
        ("n_patterns", C.c_uint32),
        ("n_species", C.c_uint32),
        ("type_patterns", C.c_void_p),
        ("chain_pattern", C.c_void_p),
        ("chiN", C.c_void_p),
        ("b", C.c_float),
        ("kappaN", C.c_float),
        ("move_halfwidth", C.c_float),
        ("smc_mobility", C.c_float),
        ("grid", C.c_uint32 * 3),
        ("reserved2", C.c_uint32),
        ("box", C.c_float * 3),
        ("reserved3", C.c_float),
        ("seed", C.c_uint64),
        ("workspace", C.c_void_p),
        ("workspace_bytes", C.c_uint64),
        ("n_single", C.c_void_p),
        ("species_n_chains", C.c_void_p),
        ("species_beads", C.c_void_p),
    ]


class soma_validation(C.Structure):
    """Mirror of `struct soma_validation` in include/soma.h."""
    _fields_ = [("n_nonfinite", C.c_uint64), ("density_total", C.c_uint64), ("density_per_type", C.c_uint64 * 8),
                ("max_bond_sq", C.c_float), ("ok", C.c_uint32), ("mean_bond_sq", C.c_double)]


_lib: Optional[C.CDLL] = None


def load_library() -> C.CDLL:
    """dlopen the in-tree libsoma_b200.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'`"
                              " (nvcc, sm_100a). There is no CPU fallback.")
        L = C.CDLL(str(LIB_PATH))
        vp, u64, u32, i32 = C.c_void_p, C.c_uint64, C.c_uint32, C.c_int
        pp = C.POINTER(soma_params)
        sig = {
            "soma_workspace_bytes": (u64, [pp]),
            "soma_create": (i32, [pp, vp, C.POINTER(vp)]),
            "soma_load_state": (i32, [vp, vp, vp, vp, u64, i32]),
            "soma_mc_steps": (i32, [vp, u32, C.POINTER(u64)]),
            "soma_get_density": (i32, [vp, vp, i32]),
            "soma_get_positions": (i32, [vp, vp, vp, vp, i32]),
            "soma_get_omega": (i32, [vp, vp, i32]),
            "soma_set_external_field": (i32, [vp, vp, i32]),
            "soma_generate_state": (i32, [vp, u64, u64]),
            "soma_init_from_density": (i32, [vp, vp, i32, u64, u64, u32, C.c_float]),
            "soma_validate_state": (i32, [vp, C.POINTER(soma_validation)]),
            "soma_validate_noalloc": (i32, [vp, vp, vp, u64, u32, vp, u32, u64, vp, C.POINTER(soma_validation), C.c_char_p, C.c_size_t]),
            "soma_get_step": (i32, [vp, C.POINTER(u64)]),
            "soma_destroy": (i32, [vp]),
            "soma_last_error": (C.c_char_p, [vp]),
            "soma_set_option": (i32, [vp, C.c_char_p, C.c_int64]),
            "soma_get_counters": (i32, [vp, C.POINTER(u64)]),
            "soma_get_kernel_times": (i32, [vp, C.POINTER(C.c_double), C.POINTER(u64)]),
            "soma_debug_half_sweep": (i32, [vp, u32, C.POINTER(u64)]),
            "soma_debug_finish_step": (i32, [vp]),
            "soma_debug_set_omega": (i32, [vp, vp]),
            "soma_debug_philox": (i32, [vp, vp, vp, u64]),
            "soma_debug_maps": (i32, [vp, vp, vp, vp, vp, u64]),
            "soma_debug_accept": (i32, [vp, vp, vp, u64]),
            "soma_debug_accept_fma": (i32, [vp, vp, vp, u64]),
            "soma_debug_cell_index": (i32, [vp, vp, vp, vp, vp, u64]),
            "soma_debug_red_throughput": (i32, [u64, u64, i32, C.POINTER(C.c_double)]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _check(rc: int, h=None):
    if rc != SOMA_OK:
        raise SomaError(rc, (load_library().soma_last_error(h) or b"").decode())


def _ptr(a) -> int:
    """Address of a numpy array (host) or torch tensor (host or device)."""
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()


def _is_device(a) -> int:
    return 0 if isinstance(a, np.ndarray) else int(a.is_cuda)


# ---- the C entry points, same names ------------------------------------------------------------

def make_params(n_chains, beads_per_chain, n_types, type_patterns, chain_pattern, b, chiN, kappaN,
                grid, box, move_halfwidth, seed, n_single=None, smc_mobility=0.0, species=None):
    """Build a soma_params plus the numpy arrays it points to (keep the tuple alive until create).
    species: None or [(n_chains_s, beads_s), ...] (soma_params.n_species, species_n_chains, species_beads)."""
    pats = np.ascontiguousarray(type_patterns, dtype=np.uint8)
    n_patterns = 1 if pats.ndim < 2 else int(pats.shape[0])     # validation is the library's job
    cp = None if chain_pattern is None else np.ascontiguousarray(chain_pattern, dtype=np.uint8)
    chi = np.ascontiguousarray(chiN, dtype=np.float32)
    p = soma_params()
    p.n_chains, p.beads_per_chain, p.n_types, p.n_patterns = int(n_chains), int(beads_per_chain), int(n_types), n_patterns
    p.type_patterns = pats.ctypes.data
    p.chain_pattern = None if cp is None else cp.ctypes.data
    p.chiN = chi.ctypes.data
    p.b, p.kappaN, p.move_halfwidth = float(b), float(kappaN), float(move_halfwidth)
    p.smc_mobility = float(smc_mobility)
    p.grid = (C.c_uint32 * 3)(*[int(g) for g in grid])
    p.box = (C.c_float * 3)(*[float(v) for v in box])
    p.seed = int(seed)
    p.workspace, p.workspace_bytes = None, 0
    ns = None if n_single is None else np.ascontiguousarray(n_single, dtype=np.uint64)
    p.n_single = None if ns is None else ns.ctypes.data
    sn = sb = None
    if species is not None:
        sn = np.ascontiguousarray([a for a, _ in species], dtype=np.uint64)
        sb = np.ascontiguousarray([c for _, c in species], dtype=np.uint32)
        p.n_species, p.species_n_chains, p.species_beads = len(species), sn.ctypes.data, sb.ctypes.data
    return p, (pats, cp, chi, ns, sn, sb)


def soma_workspace_bytes(p: soma_params) -> int:
    return int(load_library().soma_workspace_bytes(C.byref(p)))


def soma_create(p: soma_params, cuda_stream: int = 0) -> int:
    h = C.c_void_p()
    _check(load_library().soma_create(C.byref(p), C.c_void_p(cuda_stream), C.byref(h)))
    return h.value


def soma_load_state(h, x, y, z, step0: int = 0):
    dev = _is_device(x)
    assert _is_device(y) == dev and _is_device(z) == dev
    _check(load_library().soma_load_state(h, _ptr(x), _ptr(y), _ptr(z), int(step0), dev), h)


def soma_mc_steps(h, n_steps: int, want_accepted: bool = False) -> Optional[int]:
    acc = C.c_uint64(0)
    _check(load_library().soma_mc_steps(h, int(n_steps), C.byref(acc) if want_accepted else None), h)
    return int(acc.value) if want_accepted else None


def soma_get_density(h, out):
    _check(load_library().soma_get_density(h, _ptr(out), _is_device(out)), h)
    return out


def soma_get_positions(h, x, y, z):
    dev = _is_device(x)
    _check(load_library().soma_get_positions(h, _ptr(x), _ptr(y), _ptr(z), dev), h)
    return x, y, z


def soma_get_omega(h, out):
    _check(load_library().soma_get_omega(h, _ptr(out), _is_device(out)), h)
    return out


def soma_set_external_field(h, ext):
    """ext: [T][cells] fp32 numpy array or CUDA tensor, or None to remove the field."""
    if ext is None:
        _check(load_library().soma_set_external_field(h, None, 0), h)
        return
    if isinstance(ext, np.ndarray):
        ext = np.ascontiguousarray(ext, dtype=np.float32)
    _check(load_library().soma_set_external_field(h, _ptr(ext), _is_device(ext)), h)


def soma_generate_state(h, gen_seed: int, step0: int = 0):
    _check(load_library().soma_generate_state(h, int(gen_seed), int(step0)), h)


def soma_init_from_density(h, phi_target, gen_seed: int, step0: int = 0, n_equil_steps: int = 0, umbrella_k: float = 0.0):
    """phi_target: [T][cells] fp32 numpy array or CUDA tensor."""
    if isinstance(phi_target, np.ndarray):
        phi_target = np.ascontiguousarray(phi_target, dtype=np.float32)
    _check(load_library().soma_init_from_density(h, _ptr(phi_target), _is_device(phi_target), int(gen_seed), int(step0),
                                                 int(n_equil_steps), float(umbrella_k)), h)


def soma_validate_state(h) -> dict:
    v = soma_validation()
    _check(load_library().soma_validate_state(h, C.byref(v)), h)
    return {"nonfinite": int(v.n_nonfinite), "density_total": int(v.density_total),
            "density_per_type": [int(t) for t in v.density_per_type], "max_bond_sq": float(v.max_bond_sq),
            "mean_bond_sq": float(v.mean_bond_sq), "ok": bool(v.ok)}


def soma_validate_noalloc(x, y, z, n_chains: int, beads_per_chain: int, counts=None, n_types: int = 0, cells: int = 0,
                          cuda_stream: int = 0) -> dict:
    """Validation report of a state held in CUDA tensors, for callers that must not allocate device memory (a
    process whose HBM is already spoken for, a loop that cannot afford cudaMalloc's device-wide stall, a check
    made before any handle exists): the library keeps its partial results in a fixed 1.6 MB array of its own.
    x, y, z: float32 CUDA tensors of n_chains * beads_per_chain elements; counts: uint32/int32 CUDA tensor
    [n_types][cells] or None.  At most 2^28 beads per call; calls must not overlap on the GPU.  Same keys as
    soma_validate_state.  This wrapper only marshals the arguments; it creates no tensor."""
    v = soma_validation()
    err = C.create_string_buffer(512)
    rc = load_library().soma_validate_noalloc(_ptr(x), _ptr(y), _ptr(z), int(n_chains), int(beads_per_chain),
                                              None if counts is None else _ptr(counts), int(n_types), int(cells),
                                              C.c_void_p(cuda_stream), C.byref(v), err, len(err))
    if rc != SOMA_OK:
        raise SomaError(rc, err.value.decode())
    return {"nonfinite": int(v.n_nonfinite), "density_total": int(v.density_total),
            "density_per_type": [int(t) for t in v.density_per_type], "max_bond_sq": float(v.max_bond_sq),
            "mean_bond_sq": float(v.mean_bond_sq), "ok": bool(v.ok)}


def soma_get_step(h) -> int:
    s = C.c_uint64(0)
    _check(load_library().soma_get_step(h, C.byref(s)), h)
    return int(s.value)


def soma_destroy(h):
    _check(load_library().soma_destroy(h))


def soma_set_option(h, name: str, value: int):
    _check(load_library().soma_set_option(h, name.encode(), int(value)), h)


def soma_get_counters(h) -> dict:
    out = (C.c_uint64 * 6)()
    _check(load_library().soma_get_counters(h, out), h)
    return {"launches": int(out[0]), "steps": int(out[1]), "resorts": int(out[2]), "path": int(out[3]),
            "packed_counts": bool(out[4]), "omega_otf": bool(out[5])}


def soma_get_kernel_times(h) -> dict:
    ms = (C.c_double * 2)()
    n = C.c_uint64(0)
    _check(load_library().soma_get_kernel_times(h, ms, C.byref(n)), h)
    return {"move_bin_ms": float(ms[0]), "omega_ms": float(ms[1]), "steps": int(n.value)}


def soma_debug_half_sweep(h, parity: int, want_accepted: bool = True):
    acc = C.c_uint64(0)
    _check(load_library().soma_debug_half_sweep(h, int(parity), C.byref(acc) if want_accepted else None), h)
    return int(acc.value)


def soma_debug_finish_step(h):
    _check(load_library().soma_debug_finish_step(h), h)


def soma_debug_set_omega(h, omega: np.ndarray):
    omega = np.ascontiguousarray(omega, dtype=np.float32)
    _check(load_library().soma_debug_set_omega(h, omega.ctypes.data), h)


def soma_debug_philox(ctr: np.ndarray, key: Sequence[int]) -> np.ndarray:
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty_like(ctr)
    _check(load_library().soma_debug_philox(ctr.ctypes.data, k.ctypes.data, out.ctypes.data, ctr.shape[0]))
    return out


def soma_debug_maps(words: np.ndarray):
    words = np.ascontiguousarray(words, dtype=np.uint32).reshape(-1)
    t, u, l, lf = (np.empty(words.size, dtype=np.float32) for _ in range(4))
    _check(load_library().soma_debug_maps(words.ctypes.data, t.ctypes.data, u.ctypes.data, l.ctypes.data, lf.ctypes.data, words.size))
    return t, u, l, lf


def soma_debug_accept(dE: np.ndarray, words: np.ndarray) -> np.ndarray:
    dE = np.ascontiguousarray(dE, dtype=np.float32).reshape(-1)
    words = np.ascontiguousarray(words, dtype=np.uint32).reshape(-1)
    assert dE.size == words.size
    out = np.empty(dE.size, dtype=np.uint8)
    _check(load_library().soma_debug_accept(dE.ctypes.data, words.ctypes.data, out.ctypes.data, dE.size))
    return out


def soma_debug_accept_fma(dE: np.ndarray, words: np.ndarray) -> np.ndarray:
    dE = np.ascontiguousarray(dE, dtype=np.float32).reshape(-1)
    words = np.ascontiguousarray(words, dtype=np.uint32).reshape(-1)
    assert dE.size == words.size
    out = np.empty(dE.size, dtype=np.uint8)
    _check(load_library().soma_debug_accept_fma(dE.ctypes.data, words.ctypes.data, out.ctypes.data, dE.size))
    return out


def soma_debug_cell_index(h, x, y, z) -> np.ndarray:
    x, y, z = (np.ascontiguousarray(v, dtype=np.float32).reshape(-1) for v in (x, y, z))
    out = np.empty(x.size, dtype=np.uint32)
    _check(load_library().soma_debug_cell_index(h, x.ctypes.data, y.ctypes.data, z.ctypes.data, out.ctypes.data, x.size), h)
    return out


def soma_debug_red_throughput(n_counters: int, n_ops: int, mode: int) -> float:
    """milliseconds of the best of three launches; see include/soma.h"""
    ms = C.c_double(0.0)
    _check(load_library().soma_debug_red_throughput(int(n_counters), int(n_ops), int(mode), C.byref(ms)))
    return float(ms.value)


# ---- convenience wrapper -----------------------------------------------------------------------

class Soma:
    """One SCMF system on the current CUDA device.  Device memory and stream come from PyTorch."""

    def __init__(self, n_chains, beads_per_chain, n_types, type_patterns, chain_pattern, b, chiN,
                 kappaN, grid, box, move_halfwidth, seed, stream=None, lend_workspace: bool = True, n_single=None, smc_mobility=0.0,
                 species=None, workspace_fill: Optional[int] = None):
        import torch
        if not torch.cuda.is_available():
            raise SomaError(SOMA_ECUDA, "no CUDA device: this package has no CPU fallback")
        self.n_chains, self.N, self.T = int(n_chains), int(beads_per_chain), int(n_types)
        chain_beads = self.n_chains * self.N if species is None else sum(int(a) * int(c) for a, c in species)
        self.B = chain_beads + (0 if n_single is None else int(np.asarray(n_single, dtype=np.uint64).sum()))
        self.grid = tuple(int(g) for g in grid)
        self.cells = self.grid[0] * self.grid[1] * self.grid[2]
        p, keep = make_params(n_chains, beads_per_chain, n_types, type_patterns, chain_pattern, b, chiN,
                              kappaN, grid, box, move_halfwidth, seed, n_single=n_single, smc_mobility=smc_mobility, species=species)
        self._workspace = None
        if lend_workspace:
            nbytes = soma_workspace_bytes(p)
            if nbytes == 0:
                raise SomaError(SOMA_EINVAL, (load_library().soma_last_error(None) or b"").decode())
            self._workspace = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
            if workspace_fill is not None:      # tests: the library must not depend on what the lent memory holds
                self._workspace.fill_(int(workspace_fill))
            p.workspace, p.workspace_bytes = self._workspace.data_ptr(), nbytes
        self._stream = stream if stream is not None else torch.cuda.current_stream()
        self._h = soma_create(p, self._stream.cuda_stream)
        del keep

    @classmethod
    def from_system(cls, s, **kw) -> "Soma":
        """`s` is a scmf_inputs.System (duck-typed)."""
        w = s.workload
        kw.setdefault("n_single", getattr(s, "n_single", None))
        kw.setdefault("species", getattr(s, "species", None))
        return cls(w.n_chains, w.N, w.n_types, s.type_patterns, s.chain_pattern, w.b, s.chiN,
                   w.kappaN, w.grid, w.box, w.move_halfwidth, w.seed, **kw)

    def close(self):
        if getattr(self, "_h", None):
            soma_destroy(self._h)
            self._h = None
            self._workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def load_state(self, x, y, z, step0: int = 0):
        soma_load_state(self._h, x, y, z, step0)

    def generate_state(self, gen_seed: int, step0: int = 0):
        soma_generate_state(self._h, gen_seed, step0)

    def init_from_density(self, phi_target, gen_seed: int, step0: int = 0, n_equil_steps: int = 0, umbrella_k: float = 0.0):
        soma_init_from_density(self._h, phi_target, gen_seed, step0, n_equil_steps, umbrella_k)

    def validate(self) -> dict:
        return soma_validate_state(self._h)

    def mc_steps(self, n: int, want_accepted: bool = False):
        return soma_mc_steps(self._h, n, want_accepted)

    def positions(self):
        x, y, z = (np.empty(self.B, dtype=np.float32) for _ in range(3))
        return soma_get_positions(self._h, x, y, z)

    def positions_device(self):
        import torch
        x, y, z = (torch.empty(self.B, dtype=torch.float32, device="cuda") for _ in range(3))
        return soma_get_positions(self._h, x, y, z)

    def density(self) -> np.ndarray:
        return soma_get_density(self._h, np.empty((self.T, self.cells), dtype=np.uint32))

    def omega(self) -> np.ndarray:
        return soma_get_omega(self._h, np.empty((self.T, self.cells), dtype=np.float32))

    def set_external_field(self, ext):
        soma_set_external_field(self._h, ext)

    @property
    def step(self) -> int:
        return soma_get_step(self._h)

    def set_option(self, name: str, value: int):
        soma_set_option(self._h, name, value)

    def counters(self) -> dict:
        return soma_get_counters(self._h)

    def kernel_times(self) -> dict:
        return soma_get_kernel_times(self._h)

    # test hooks
    def debug_half_sweep(self, parity: int) -> int:
        return soma_debug_half_sweep(self._h, parity)

    def debug_finish_step(self):
        soma_debug_finish_step(self._h)

    def debug_set_omega(self, omega):
        soma_debug_set_omega(self._h, omega)

    def debug_cell_index(self, x, y, z):
        return soma_debug_cell_index(self._h, x, y, z)
