"""ctypes driver for the CPU oracle (oracle/scmf_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this package.  It never imports paper_2606_09356_b200 and shares no code with it.
Argument marshalling only: every number the oracle produces is computed in scmf_oracle.cpp.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "scmf_oracle.cpp"
_LIB = _HERE / "libscmf_oracle.so"

# -ffp-contract=off: an FMA appears only where the source writes fmaf() (R17).
_CXXFLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
             "-Wall", "-Wextra"]


def _isa_flags():
    """-mfma/-msse4.1 when the host has them: fmaf()/floorf() become one instruction instead of a
    libm call.  Results are identical either way (both are the IEEE fused multiply-add / floor)."""
    try:
        flags = set()
        for line in open("/proc/cpuinfo"):
            if line.startswith("flags"):
                flags = set(line.split(":", 1)[1].split())
                break
        return [f for f, need in (("-mfma", "fma"), ("-msse4.1", "sse4_1")) if need in flags]
    except OSError:
        return []


# SCMF_ORACLE_SANITIZE=1 (tests/test_oracle_sanitizers.py): the same source, instrumented with AddressSanitizer and
# UndefinedBehaviorSanitizer, as a second library.  The process must then run with libasan preloaded.  Same flags
# otherwise (-O2, no contraction), so the instrumented oracle computes the same bits.
_SAN_LIB = _HERE / "libscmf_oracle_san.so"
_SAN_FLAGS = ["-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined,float-cast-overflow,float-divide-by-zero",
              "-fno-sanitize-recover=all"]


def sanitized() -> bool:
    return os.environ.get("SCMF_ORACLE_SANITIZE", "") == "1"


def build(force: bool = False) -> Path:
    """Compile the oracle with g++ (no GPU involved).  Returns the path of the shared library."""
    out, extra = (_SAN_LIB, _SAN_FLAGS) if sanitized() else (_LIB, [])
    if force or not out.exists() or out.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = out.with_suffix(f".tmp{os.getpid()}.so")
        subprocess.run(["g++", *_CXXFLAGS, *extra, *_isa_flags(), str(_SRC), "-o", str(tmp)], check=True)
        os.replace(tmp, out)
    return out


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        u8p, u32p, u64p = C.POINTER(C.c_uint8), C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
        f32p, f64p, vp = C.POINTER(C.c_float), C.POINTER(C.c_double), C.c_void_p
        sig = {
            "oracle_philox4x32_10": (None, [u32p, u32p, u32p]),
            "oracle_tmap": (C.c_float, [C.c_uint32]),
            "oracle_umap": (C.c_float, [C.c_uint32]),
            "oracle_lnu": (C.c_float, [C.c_float]),
            "oracle_lnu_array": (None, [f32p, f32p, C.c_uint64]),
            "oracle_create": (vp, [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, u8p, u8p,
                                   C.c_float, f32p, C.c_float, u32p, f32p, C.c_float, C.c_uint64]),
            "oracle_destroy": (None, [vp]),
            "oracle_load_state": (C.c_int, [vp, f32p, f32p, f32p, C.c_uint64]),
            "oracle_mc_steps": (C.c_uint64, [vp, C.c_uint32]),
            "oracle_half_sweep": (C.c_uint64, [vp, C.c_uint32, C.c_int, u64p, C.c_uint64, u8p, f64p]),
            "oracle_bin": (None, [vp]),
            "oracle_compute_omega": (None, [vp]),
            "oracle_finish_step": (None, [vp]),
            "oracle_get_positions": (None, [vp, f32p, f32p, f32p]),
            "oracle_set_beads": (None, [vp, u64p, C.c_uint64, f32p, f32p, f32p]),
            "oracle_get_density": (None, [vp, u32p]),
            "oracle_set_density": (None, [vp, u32p]),
            "oracle_get_omega": (None, [vp, f32p]),
            "oracle_set_omega": (None, [vp, f32p]),
            "oracle_set_external_field": (None, [vp, f32p]),
            "oracle_generate_state": (C.c_int, [vp, C.c_uint64, C.c_uint64]),
            "oracle_init_from_density": (C.c_int, [vp, f32p, C.c_uint64, C.c_uint64]),
            "oracle_set_umbrella": (None, [vp, f32p, C.c_float]),
            "oracle_set_singles": (C.c_int, [vp, C.POINTER(C.c_uint64)]),
            "oracle_set_species": (C.c_int, [vp, C.c_uint32, C.POINTER(C.c_uint64), C.POINTER(C.c_uint32), C.c_uint32]),
            "oracle_set_smc": (None, [vp, C.c_float]),
            "oracle_smc_margin": (C.c_float, [vp, C.c_uint64, C.c_float, C.c_float, C.c_float]),
            "oracle_smc_draws": (None, [vp, C.c_uint64, C.c_uint32, C.c_uint32, C.POINTER(C.c_double)]),
            "oracle_det_functions": (None, [C.c_double, C.POINTER(C.c_double)]),
            "oracle_det_functions_n": (None, [f32p, C.c_uint64, f32p, f32p, f32p]),
            "oracle_validate": (None, [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_double)]),
            "oracle_get_step": (C.c_uint64, [vp]),
            "oracle_set_step": (None, [vp, C.c_uint64]),
            "oracle_cell_index": (C.c_uint64, [vp, C.c_float, C.c_float, C.c_float]),
            "oracle_delta_energy": (C.c_float, [vp, C.c_uint64, C.c_float, C.c_float, C.c_float]),
            "oracle_trial": (None, [vp, C.c_uint64, C.c_uint32, f32p, f32p]),
            "oracle_get_constants": (None, [vp, f32p]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _p(a: np.ndarray, ctype):
    return a.ctypes.data_as(C.POINTER(ctype))


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def tmap(w: int) -> float:
    return float(lib().oracle_tmap(int(w) & 0xFFFFFFFF))


def umap(w: int) -> float:
    return float(lib().oracle_umap(int(w) & 0xFFFFFFFF))


def lnu(u) -> np.ndarray:
    u = np.ascontiguousarray(u, dtype=np.float32).reshape(-1)
    out = np.empty_like(u)
    lib().oracle_lnu_array(_p(u, C.c_float), _p(out, C.c_float), u.size)
    return out


def det_functions(x: float):
    """(det_log(x), sin(2 pi x), cos(2 pi x)) of the library-free routines behind the normal deviates (R24)."""
    out = (C.c_double * 3)()
    lib().oracle_det_functions(float(x), out)
    return float(out[0]), float(out[1]), float(out[2])


def det_functions_n(x: np.ndarray):
    """det_functions over an array of fp32 arguments: (log, sin 2 pi x, cos 2 pi x) as fp32 arrays."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    lg, sn, cs = (np.empty(x.size, dtype=np.float32) for _ in range(3))
    lib().oracle_det_functions_n(_p(x, C.c_float), x.size, _p(lg, C.c_float), _p(sn, C.c_float), _p(cs, C.c_float))
    return lg, sn, cs


class Oracle:
    """One SCMF system held by the CPU oracle."""

    def __init__(self, n_chains, N, n_types, type_patterns, chain_pattern, b, chiN, kappaN,
                 grid, box, move_halfwidth, seed, n_single=None, species=None):
        """species: None, or [(n_chains_s, N_s), ...] -- polymer species of different chain lengths stored one
        after the other (R26); N is then the reference chain length of 1/N and the pattern rows have
        max N_s entries."""
        self.n_chains, self.N, self.T = int(n_chains), int(N), int(n_types)
        self.species = None if species is None else [(int(a), int(b_)) for a, b_ in species]
        stride = self.N if species is None else max(ns for _, ns in self.species)
        self.B = self.n_chains * self.N if species is None else sum(a * b_ for a, b_ in self.species)
        self.grid = tuple(int(g) for g in grid)
        self.Cells = self.grid[0] * self.grid[1] * self.grid[2]
        pats = np.ascontiguousarray(type_patterns, dtype=np.uint8).reshape(-1, stride)
        cp = None if chain_pattern is None else np.ascontiguousarray(chain_pattern, dtype=np.uint8)
        chi = np.ascontiguousarray(chiN, dtype=np.float32).reshape(self.T, self.T)
        g = np.asarray(self.grid, dtype=np.uint32)
        bx = np.asarray(box, dtype=np.float32)
        self._h = lib().oracle_create(
            self.n_chains, stride, self.T, pats.shape[0], _p(pats, C.c_uint8),
            None if cp is None else _p(cp, C.c_uint8), float(b), _p(chi, C.c_float),
            float(kappaN), _p(g, C.c_uint32), _p(bx, C.c_float), float(move_halfwidth), int(seed))
        if not self._h:
            raise ValueError("oracle_create rejected the parameters")
        if species is not None:
            assert sum(a for a, _ in self.species) == self.n_chains
            cnt = np.array([a for a, _ in self.species], dtype=np.uint64)
            lens = np.array([b_ for _, b_ in self.species], dtype=np.uint32)
            if lib().oracle_set_species(self._h, len(self.species), _p(cnt, C.c_uint64), _p(lens, C.c_uint32), self.N) != 0:
                raise ValueError("oracle_set_species rejected the species table")
        if n_single is not None:                     # single-bead molecules per type, stored after the chains (R23)
            ns = np.ascontiguousarray(n_single, dtype=np.uint64).reshape(self.T)
            if lib().oracle_set_singles(self._h, _p(ns, C.c_uint64)) != 0:
                raise ValueError("too many molecules")
            self.B += int(ns.sum())

    @classmethod
    def from_system(cls, s) -> "Oracle":
        """`s` is a scmf_inputs.System (duck-typed; this package imports nothing of it)."""
        w = s.workload
        return cls(w.n_chains, w.N, w.n_types, s.type_patterns, s.chain_pattern, w.b, s.chiN,
                   w.kappaN, w.grid, w.box, w.move_halfwidth, w.seed, n_single=getattr(s, "n_single", None),
                   species=getattr(s, "species", None))

    def close(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    __del__ = close

    def load_state(self, x, y, z, step0: int = 0):
        x, y, z = (np.ascontiguousarray(v, dtype=np.float32) for v in (x, y, z))
        assert x.size == y.size == z.size == self.B
        lib().oracle_load_state(self._h, _p(x, C.c_float), _p(y, C.c_float), _p(z, C.c_float), int(step0))

    def generate_state(self, gen_seed: int, step0: int = 0):
        """Gaussian random-walk initial state by the recipe of DESIGN.md R22, then bin + omega."""
        lib().oracle_generate_state(self._h, int(gen_seed), int(step0))

    def init_from_density(self, phi_target, gen_seed: int, step0: int = 0, n_equil_steps: int = 0, umbrella_k: float = 0.0) -> int:
        """Initial state reproducing the target concentrations phi_target [T][C] (R25), then
        n_equil_steps MC steps under the umbrella potential of strength umbrella_k, which is removed again.
        Returns the number of moves accepted during the equilibration."""
        phi = np.ascontiguousarray(phi_target, dtype=np.float32).reshape(self.T, self.Cells)
        rc = lib().oracle_init_from_density(self._h, _p(phi, C.c_float), int(gen_seed), int(step0))
        if rc != 0:
            raise ValueError({-1: "phi_target holds a negative, NaN or too large value", -2: "a species has zero total target weight"}[rc])
        acc = 0
        if n_equil_steps:
            self.set_umbrella(phi, umbrella_k)
            acc = self.mc_steps(n_equil_steps)
            self.set_umbrella(None, 0.0)
        return acc

    def set_umbrella(self, phi_target, k: float):
        """Umbrella potential toward phi_target [T][C] with strength k (R25); None switches it off."""
        if phi_target is None:
            lib().oracle_set_umbrella(self._h, None, 0.0)
        else:
            phi = np.ascontiguousarray(phi_target, dtype=np.float32).reshape(self.T, self.Cells)
            lib().oracle_set_umbrella(self._h, _p(phi, C.c_float), float(k))

    def set_smc(self, A: float):
        """A > 0: bond-force-biased moves with mobility A (R24); 0: uniform moves."""
        lib().oracle_set_smc(self._h, float(A))

    def smc_margin(self, bead: int, nx, ny, nz) -> float:
        return float(lib().oracle_smc_margin(self._h, int(bead), float(nx), float(ny), float(nz)))

    def smc_draws(self, chain: int, bead: int, parity: int):
        out = (C.c_double * 4)()
        lib().oracle_smc_draws(self._h, int(chain), int(bead), int(parity), out)
        return [float(v) for v in out]

    def validate(self) -> dict:
        """Non-finite coordinates, density totals, largest and mean squared bond length of the state."""
        out = (C.c_uint64 * 10)()
        bond = (C.c_double * 2)()
        lib().oracle_validate(self._h, out, bond)
        return {"nonfinite": int(out[0]), "density_total": int(out[1]), "density_per_type": [int(out[2 + t]) for t in range(self.T)],
                "max_bond_sq": float(bond[0]), "mean_bond_sq": float(bond[1])}

    def mc_steps(self, n: int) -> int:
        return int(lib().oracle_mc_steps(self._h, int(n)))

    def half_sweep(self, parity: int, order: int = 0, perm=None, want_mask=False, want_margins=False):
        mask = np.zeros(self.B, dtype=np.uint8) if want_mask else None
        marg = np.full(self.B, np.nan, dtype=np.float64) if want_margins else None
        pp, n_perm = None, 0
        if perm is not None:
            perm = np.ascontiguousarray(perm, dtype=np.uint64)
            pp, n_perm = _p(perm, C.c_uint64), perm.size
        acc = int(lib().oracle_half_sweep(
            self._h, int(parity), int(order), pp, n_perm,
            None if mask is None else _p(mask, C.c_uint8),
            None if marg is None else _p(marg, C.c_double)))
        return acc, mask, marg

    def bin(self):
        lib().oracle_bin(self._h)

    def compute_omega(self):
        lib().oracle_compute_omega(self._h)

    def finish_step(self):
        lib().oracle_finish_step(self._h)

    def positions(self):
        x, y, z = (np.empty(self.B, dtype=np.float32) for _ in range(3))
        lib().oracle_get_positions(self._h, _p(x, C.c_float), _p(y, C.c_float), _p(z, C.c_float))
        return x, y, z

    def set_beads(self, idx, x, y, z):
        idx = np.ascontiguousarray(idx, dtype=np.uint64)
        x, y, z = (np.ascontiguousarray(v, dtype=np.float32) for v in (x, y, z))
        lib().oracle_set_beads(self._h, _p(idx, C.c_uint64), idx.size, _p(x, C.c_float),
                               _p(y, C.c_float), _p(z, C.c_float))

    def density(self) -> np.ndarray:
        out = np.empty((self.T, self.Cells), dtype=np.uint32)
        lib().oracle_get_density(self._h, _p(out, C.c_uint32))
        return out

    def set_density(self, counts):
        counts = np.ascontiguousarray(counts, dtype=np.uint32).reshape(self.T, self.Cells)
        lib().oracle_set_density(self._h, _p(counts, C.c_uint32))

    def omega(self) -> np.ndarray:
        out = np.empty((self.T, self.Cells), dtype=np.float32)
        lib().oracle_get_omega(self._h, _p(out, C.c_float))
        return out

    def set_omega(self, omega):
        omega = np.ascontiguousarray(omega, dtype=np.float32).reshape(self.T, self.Cells)
        lib().oracle_set_omega(self._h, _p(omega, C.c_float))

    def set_external_field(self, ext):
        """ext [T][C] in kT per bead, added to omega (R21); None removes it."""
        if ext is None:
            lib().oracle_set_external_field(self._h, None)
        else:
            ext = np.ascontiguousarray(ext, dtype=np.float32).reshape(self.T, self.Cells)
            lib().oracle_set_external_field(self._h, _p(ext, C.c_float))

    @property
    def step(self) -> int:
        return int(lib().oracle_get_step(self._h))

    @step.setter
    def step(self, t: int):
        lib().oracle_set_step(self._h, int(t))

    def cell_index(self, x, y, z) -> int:
        return int(lib().oracle_cell_index(self._h, float(x), float(y), float(z)))

    def delta_energy(self, bead: int, nx, ny, nz) -> float:
        return float(lib().oracle_delta_energy(self._h, int(bead), float(nx), float(ny), float(nz)))

    def trial(self, bead: int, parity: int):
        xyz = np.zeros(3, dtype=np.float32)
        u = C.c_float(0)
        lib().oracle_trial(self._h, int(bead), int(parity), _p(xyz, C.c_float), C.byref(u))
        return xyz, np.float32(u.value)

    def constants(self) -> dict:
        out = np.zeros(6, dtype=np.float32)
        lib().oracle_get_constants(self._h, _p(out, C.c_float))
        return {"kb": out[0], "inv_h": out[1:4].copy(), "dens_scale": out[4], "invN": out[5]}
