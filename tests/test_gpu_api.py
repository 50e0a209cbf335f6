"""Behaviour of the C ABI on a device: call ordering, error codes, host/device pointers, lent and
library-owned workspaces, streams, and the checkpoint invariant (the random
stream is keyed by the absolute step, so (positions, step) is a complete checkpoint)."""
import ctypes as C

import numpy as np
import pytest

import oracle
import scmf_inputs as si
from helpers import assert_same_state, gpu_system

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def soma():
    import __graft_entry__ as entry
    entry.build()
    import paper_2606_09356_b200 as soma
    return soma


@pytest.fixture(scope="module")
def small():
    return si.make_system(si.scaled(si.config(2), 2050, (8, 8, 8)))


def test_call_order_and_error_codes(soma, small):
    s = small
    lib = soma.load_library()
    with gpu_system(s) as g:
        h = g._h
        assert lib.soma_mc_steps(h, 1, None) == soma.SOMA_ESTATE
        assert b"load_state" in lib.soma_last_error(h)
        dens = np.zeros((2, 512), dtype=np.uint32)
        assert lib.soma_get_density(h, dens.ctypes.data, 0) == soma.SOMA_ESTATE
        assert lib.soma_get_positions(h, None, None, None, 0) == soma.SOMA_EINVAL
        assert lib.soma_load_state(h, None, s.y.ctypes.data, s.z.ctypes.data, 0, 0) == soma.SOMA_EINVAL
        assert lib.soma_load_state(h, s.x.ctypes.data, s.y.ctypes.data, s.z.ctypes.data, 1 << 48, 0) == soma.SOMA_EINVAL
        assert lib.soma_set_option(h, b"no_such_option", 1) == soma.SOMA_EINVAL
        assert lib.soma_set_option(h, b"path", 7) == soma.SOMA_EINVAL
        g.load_state(s.x, s.y, s.z)
        assert g.mc_steps(0, want_accepted=True) == 0           # n_steps == 0 is a no-op
        assert g.step == 0
        assert lib.soma_debug_half_sweep(h, 2, None) == soma.SOMA_EINVAL
        g.mc_steps(1)
        assert g.step == 1
    assert lib.soma_destroy(None) == soma.SOMA_OK


def test_lent_workspace_too_small_or_misaligned(soma, small):
    import torch
    s, w = small, small.workload
    p, keep = soma.make_params(w.n_chains, w.N, w.n_types, s.type_patterns, s.chain_pattern, w.b, s.chiN, w.kappaN,
                               w.grid, w.box, w.move_halfwidth, w.seed)
    need = soma.soma_workspace_bytes(p)
    buf = torch.empty(need + 512, dtype=torch.uint8, device="cuda")
    base = (buf.data_ptr() + 255) // 256 * 256
    p.workspace, p.workspace_bytes = base, need - 1
    with pytest.raises(soma.SomaError) as e:
        soma.soma_create(p, 0)
    assert e.value.code == soma.SOMA_ENOMEM
    p.workspace, p.workspace_bytes = base + 4, need
    with pytest.raises(soma.SomaError) as e:
        soma.soma_create(p, 0)
    assert e.value.code == soma.SOMA_ENOMEM
    p.workspace, p.workspace_bytes = base, need
    h = soma.soma_create(p, 0)
    soma.soma_destroy(h)


@pytest.mark.parametrize("lend", [True, False])
def test_owned_and_lent_workspace_give_the_same_result(small, lend):
    s = small
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    o.mc_steps(3)
    with gpu_system(s, lend_workspace=lend) as g:
        g.load_state(s.x, s.y, s.z)
        g.mc_steps(3)
        assert_same_state(g, o, f"lend_workspace={lend}")


def test_device_pointers_in_and_out_and_side_stream(soma, small):
    import torch
    s = small
    o = oracle.Oracle.from_system(s)
    o.load_state(s.x, s.y, s.z)
    o.mc_steps(2)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        dx, dy, dz = (torch.from_numpy(v).cuda() for v in (s.x, s.y, s.z))
        stream.synchronize()
        with gpu_system(s, stream=stream) as g:
            g.load_state(dx, dy, dz)
            g.mc_steps(2)
            ox, oy, oz = g.positions_device()
            dens = torch.empty((2, g.cells), dtype=torch.int32, device="cuda")
            soma.soma_get_density(g._h, dens)
            om = torch.empty((2, g.cells), dtype=torch.float32, device="cuda")
            soma.soma_get_omega(g._h, om)
            stream.synchronize()
            wx, wy, wz = o.positions()
            assert np.array_equal(ox.cpu().numpy(), wx) and np.array_equal(oy.cpu().numpy(), wy) and np.array_equal(oz.cpu().numpy(), wz)
            assert np.array_equal(dens.cpu().numpy().view(np.uint32), o.density())
            assert np.array_equal(om.cpu().numpy().view(np.uint32), o.omega().view(np.uint32))
            # the caller's input tensors were copied, not adopted
            assert np.array_equal(dx.cpu().numpy(), s.x)


@pytest.mark.parametrize("path", [1, 2])
def test_checkpoint_invariance(small, path):
    """mc_steps(10) == 10 x mc_steps(1) == mc_steps(4), get, load into a NEW handle, mc_steps(6)."""
    s = small

    def final(plan):
        with gpu_system(s, path=path) as g:
            g.load_state(s.x, s.y, s.z, 100)
            acc = sum(g.mc_steps(k, want_accepted=True) for k in plan)
            return acc, g.positions(), g.density(), g.omega(), g.step

    a = final([10])
    b = final([1] * 10)
    assert a[0] == b[0] and a[4] == b[4] == 110
    for u, v in zip(a[1], b[1]):
        assert np.array_equal(u, v)
    assert np.array_equal(a[2], b[2]) and np.array_equal(a[3].view(np.uint32), b[3].view(np.uint32))
    with gpu_system(s, path=path) as g:
        g.load_state(s.x, s.y, s.z, 100)
        acc = g.mc_steps(4, want_accepted=True)
        x, y, z = g.positions()
        step = g.step
    with gpu_system(s, path=3 - path) as g2:                    # resume on the OTHER kernel path
        g2.load_state(x, y, z, step)
        acc += g2.mc_steps(6, want_accepted=True)
        assert acc == a[0] and g2.step == 110
        for u, v in zip(a[1], g2.positions()):
            assert np.array_equal(u, v)
        assert np.array_equal(a[2], g2.density())


def test_two_handles_are_independent(small):
    s = small
    with gpu_system(s) as g1, gpu_system(s) as g2:
        g1.load_state(s.x, s.y, s.z)
        g2.load_state(s.x, s.y, s.z, 7)
        g1.mc_steps(2)
        g2.mc_steps(2)
        assert g1.step == 2 and g2.step == 9
        assert not np.array_equal(g1.positions()[0], g2.positions()[0])
        o = oracle.Oracle.from_system(s)
        o.load_state(s.x, s.y, s.z)
        o.mc_steps(2)
        assert_same_state(g1, o, "handle 1 next to handle 2")


def test_launch_counter_counts_kernels(small):
    s = small
    with gpu_system(s, path=2, options=dict(omega_otf=0)) as g:
        g.load_state(s.x, s.y, s.z)
        before = g.counters()
        g.mc_steps(5)
        after = g.counters()
        assert after["steps"] - before["steps"] == 5
        assert after["launches"] - before["launches"] == 5 * 2 + 3 * (after["resorts"] - before["resorts"])   # fused move+bin, omega
    with gpu_system(s, path=2, options=dict(packed_counts=1, omega_otf=1)) as g:      # omega computed inside the move kernel: one launch per step
        g.load_state(s.x, s.y, s.z)
        before = g.counters()
        g.mc_steps(5)
        assert g.counters()["launches"] - before["launches"] == 5 and g.counters()["omega_otf"] and g.counters()["packed_counts"]
        g.omega()                                                   # the array is filled when it is asked for
        assert g.counters()["launches"] - before["launches"] == 6
    with gpu_system(s, path=1) as g:
        g.load_state(s.x, s.y, s.z)
        before = g.counters()
        g.mc_steps(5)
        assert g.counters()["launches"] - before["launches"] == 5 * 4   # even, odd, bin, omega


def test_error_codes_of_the_calls_beyond_the_six(soma, small):
    s = small
    lib = soma.load_library()
    with gpu_system(s) as g:
        h = g._h
        v = soma.soma_validation()
        assert lib.soma_validate_state(h, C.byref(v)) == soma.SOMA_ESTATE          # nothing loaded yet
        assert lib.soma_validate_state(h, None) == soma.SOMA_EINVAL
        assert lib.soma_generate_state(h, 1, 1 << 48) == soma.SOMA_EINVAL
        ext = np.full((2, 512), 0.25, dtype=np.float32)
        g.set_external_field(ext)                                                   # allowed before a state exists ...
        g.load_state(s.x, s.y, s.z)
        o = oracle.Oracle.from_system(s)
        o.load_state(s.x, s.y, s.z)
        o.set_external_field(ext)
        assert np.array_equal(g.omega().view(np.uint32), o.omega().view(np.uint32))   # ... and applied by the load
    # parameter validation at create: negative mobility, too many molecules
    for bad in (dict(smc_mobility=-1.0), dict(n_single=np.array([1 << 33, 0], dtype=np.uint64))):
        with pytest.raises(soma.SomaError) as e:
            soma.Soma.from_system(s, **bad)
        assert e.value.code == soma.SOMA_EINVAL
    # bond-force-biased moves run on the general fused kernel (path 2) wherever N allows it
    with gpu_system(si.make_system(si.scaled(si.config(4), 8192, (32, 32, 32))), smc_mobility=0.05) as g:
        assert g.counters()["path"] == 2
