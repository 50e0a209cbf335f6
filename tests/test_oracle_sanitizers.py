"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (SURVEY.md section 4 "tools" row, section 5: "host
oracle under -fsanitize=address,undefined").  A second build of oracle/scmf_oracle.cpp with the instrumentation runs
every entry point the parity tests rely on -- both move types, several species and single-bead molecules, external
field and umbrella potential, generated and density-placed starts, validation, the per-move probes -- in a child
process with libasan preloaded; any out-of-bounds access, use after free, misaligned access, signed overflow, bad
shift or float-to-integer overflow aborts the child.  The instrumented library must also give the same bits as the
plain one (same -O2, no contraction), which ties the clean bill to the code the parity tests use."""
import os
import subprocess
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[1]

CHILD = r"""
import sys
import numpy as np
sys.path.insert(0, %(root)r)
import oracle
import scmf_inputs as si
assert oracle.sanitized() and oracle.build().name == "libscmf_oracle_san.so"
out = {}

s = si.make_system(si.config(0))                                  # cfg0: diblock melt, uniform moves
o = oracle.Oracle.from_system(s)
o.load_state(s.x, s.y, s.z)
out["cfg0_acc"] = o.mc_steps(2)
acc, mask, marg = o.half_sweep(0, want_mask=True, want_margins=True)
o.half_sweep(1, order=1)
o.finish_step()
out["cfg0_x"] = o.positions()[0].copy(); out["cfg0_density"] = o.density().copy(); out["cfg0_omega"] = o.omega().copy()
out["cfg0_valid"] = np.array([o.validate()["mean_bond_sq"]])
o.cell_index(-0.25, 7.99, 8.0); o.delta_energy(5, 0.1, 0.2, 0.3); o.trial(7, 1); o.constants()
ext = np.linspace(-1, 1, 2 * 16 ** 3, dtype=np.float32).reshape(2, -1)
o.set_external_field(ext); o.mc_steps(1); o.set_external_field(None)
o.set_smc(0.05); out["cfg0_smc_acc"] = o.mc_steps(2); o.smc_margin(3, 0.1, 0.2, 0.3); o.smc_draws(1, 2, 0)
out["cfg0_smc_x"] = o.positions()[0].copy()
o.close()

s = si.make_system(si.scaled(si.config(3), 301, (16, 8, 8)))     # blend: two chain patterns, odd chain count
o = oracle.Oracle.from_system(s)
o.generate_state(11, step0=3)
o.mc_steps(1)
phi = np.random.default_rng(3).uniform(0.1, 1.2, size=(2, 16 * 8 * 8)).astype(np.float32)
o.init_from_density(phi, 5, n_equil_steps=2, umbrella_k=0.7)
out["cfg3_x"] = o.positions()[0].copy(); out["cfg3_density"] = o.density().copy()
o.close()

s = si.species_system([(40, 16), (25, 5), (7, 33)], 16, 3, np.random.default_rng(1).integers(0, 3, size=(2, 33)).astype(np.uint8),
                      np.random.default_rng(2).integers(0, 2, size=72).astype(np.uint8), [[0, 5, 9], [5, 0, 2], [9, 2, 0]], 20.0,
                      (6, 5, 3), (3.0, 2.5, 1.5), seed=9, n_single=[30, 0, 11])
o = oracle.Oracle.from_system(s)
o.load_state(s.x, s.y, s.z)
out["species_acc"] = o.mc_steps(3)
out["species_x"] = o.positions()[0].copy(); out["species_density"] = o.density().copy(); out["species_omega"] = o.omega().copy()
o.validate()
o.close()

oracle.philox4x32_10([1, 2, 3, 4], [5, 6]); oracle.lnu(np.array([1.0, 2 ** -24], dtype=np.float32)); oracle.det_functions(0.3)
oracle.det_functions_n(np.linspace(0.01, 0.99, 1000, dtype=np.float32))
np.savez(sys.argv[1], **{k: np.asarray(v) for k, v in out.items()})
print("child ok")
"""


def _run_child(tmp_path, sanitize):
    env = dict(os.environ)
    out = tmp_path / ("san.npz" if sanitize else "plain.npz")
    script = CHILD % {"root": str(ROOT)}
    if sanitize:
        asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True, check=True).stdout.strip()
        env.update(SCMF_ORACLE_SANITIZE="1", LD_PRELOAD=os.path.realpath(asan),
                   ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=97", UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    else:
        script = script.replace('assert oracle.sanitized() and oracle.build().name == "libscmf_oracle_san.so"', "assert not oracle.sanitized()")
        env.pop("SCMF_ORACLE_SANITIZE", None)
    r = subprocess.run([sys.executable, "-c", script, str(out)], env=env, capture_output=True, text=True, timeout=900)
    return r, out


def test_oracle_runs_clean_under_asan_and_ubsan_and_gives_the_same_bits(tmp_path):
    r, san = _run_child(tmp_path, True)
    assert r.returncode == 0 and "child ok" in r.stdout, r.stderr[-4000:]
    assert "AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, r.stderr[-4000:]
    r2, plain = _run_child(tmp_path, False)
    assert r2.returncode == 0, r2.stderr[-2000:]
    a, b = np.load(san), np.load(plain)
    assert sorted(a.files) == sorted(b.files) and len(a.files) >= 12
    for k in a.files:
        assert a[k].dtype == b[k].dtype and np.atleast_1d(a[k]).tobytes() == np.atleast_1d(b[k]).tobytes(), k
