"""GPU: C-ABI behaviour of liblbm_b200.so -- argument checks, call-order rules, ownership."""
import ctypes as C

import numpy as np
import pytest

import paper_2112_08926_b200 as lbm
import workloads as wl

pytestmark = pytest.mark.gpu


def test_create_rejects_bad_arguments():
    for kw, code in [(dict(nx=0), lbm.E_INVAL), (dict(velset=7), lbm.E_INVAL), (dict(tau=0.5), lbm.E_INVAL),
                     (dict(ddf_format=9), lbm.E_INVAL), (dict(collision=2), lbm.E_INVAL),
                     (dict(velset=9, nz=2), lbm.E_INVAL)]:
        args = dict(nx=8, ny=8, nz=8, velset=19, ddf_format=0, tau=0.6, collision=0)
        args.update(kw)
        with pytest.raises(lbm.LbmError) as e:
            lbm.Simulation(args["nx"], args["ny"], args["nz"], args["velset"], args["ddf_format"], args["tau"],
                           collision=args["collision"])
        assert e.value.code == code
        assert lbm.last_error()


def test_call_order_and_flags_validation():
    s = lbm.Simulation(8, 4, 4, 19, "FP16S", 0.6)
    with pytest.raises(lbm.LbmError) as e:
        s.step(1)
    assert e.value.code == lbm.E_STATE
    with pytest.raises(lbm.LbmError) as e:
        s.set_flags(np.full(128, 8, np.uint8))
    assert e.value.code == lbm.E_INVAL
    s.init(np.ones(128, np.float32), np.zeros((3, 128), np.float32))
    with pytest.raises(lbm.LbmError) as e:
        s.set_flags(np.zeros(128, np.uint8))
    assert e.value.code == lbm.E_STATE
    with pytest.raises(lbm.LbmError):
        s.step(-1)
    s.step(0)
    assert s.steps_done == 0
    s.step(3)
    assert s.steps_done == 3
    rho, u = s.read_rho_u()
    assert np.all(rho == 1.0) and np.all(u == 0.0)          # rest state is a fixed point
    for i in range(19):
        assert np.all((s.read_ddf(i) & 0x7FFF) == 0)        # codes 0x0000 / 0x8000 only
    s.close()


def test_library_owned_memory_and_device_io_agree_with_torch_memory():
    import torch
    w = wl.perturbed_equilibrium(20, 6, 4, seed=2)
    a = lbm.from_workload(w, "FP16C")                       # torch-owned DDF buffers, host init
    b = lbm.Simulation(w.nx, w.ny, w.nz, 19, "FP16C", w.tau, use_torch_memory=False)
    b.init(torch.from_numpy(w.rho).cuda(), torch.from_numpy(w.u).cuda())   # library-owned, device init
    a.step(7)
    b.step(7)
    ra, ua = a.read_rho_u()
    rb, ub = b.read_rho_u_device()
    assert np.array_equal(ra, rb.cpu().numpy()) and np.array_equal(ua, ub.cpu().numpy())


def test_launch_counter_counts_kernels():
    w = wl.perturbed_equilibrium(16, 4, 4, seed=2)
    s = lbm.from_workload(w, "FP32")
    n0 = lbm.launch_count()
    s.step(5)
    assert lbm.launch_count() - n0 == 5


def test_sizes():
    assert lbm.bytes_per_cell(19, "FP32") == 153 and lbm.bytes_per_cell(19, "FP16S") == 77
    assert lbm.bytes_per_cell(27, "FP32") == 217 and lbm.bytes_per_cell(9, "P16_2C") == 37
    assert lbm.ddf_buffer_bytes(32, 32, 32, 19, "FP16C") == 32 ** 3 * 19 * 2


def test_read_rho_u_at_equals_full_readout():
    import workloads as wl
    w = wl.perturbed_equilibrium(32, 6, 5, seed=9)
    w = wl.random_walls(w, 0.1, seed=2, moving_fraction=0.5)
    w.force = (1e-5, 0.0, 2e-5)
    for name in ("FP32", "FP16C"):
        s = lbm.from_workload(w, name)
        s.step(7)
        rho, u = s.read_rho_u()
        cells = np.array([0, 5, 31, 32, 500, w.n_cells - 1, 77], np.int64)
        r, v = s.read_rho_u_at(cells)
        assert np.array_equal(r.view(np.uint32), rho[cells].view(np.uint32))
        assert np.array_equal(v.view(np.uint32), u[:, cells].view(np.uint32))
        with pytest.raises(lbm.LbmError):
            s.read_rho_u_at([w.n_cells])
        s.close()


def test_no_write_outside_the_bound_ddf_buffers():
    """compute-sanitizer is closed on this pool: the DDF buffers are bound inside a larger tensor filled with a
    canary pattern, and the canaries must survive init, steps and read-out of both kernels on ragged shapes."""
    import ctypes as C

    import torch

    import workloads as wl
    L = lbm.lib()
    guard = 1 << 16
    for q, shape in ((19, (48, 5, 3)), (19, (1040, 2, 2)), (27, (32, 3, 3)), (9, (64, 7, 1)), (19, (37, 3, 2))):
        w = wl.perturbed_equilibrium(*shape, seed=8, velset=q)
        w = wl.random_walls(w, 0.1, seed=3, moving_fraction=0.5)
        for name in ("FP32", "FP16S", "P16_2C"):
            for variant in (2 if shape[0] % 2 == 0 else 1, lbm.VARIANT_STAGED):
                if variant >= 16 and shape[0] % 16:
                    continue
                nb = lbm.ddf_buffer_bytes(*shape, q, name)
                big = torch.full((2 * nb + 3 * guard,), 0xA5, dtype=torch.uint8, device="cuda")
                a = big.data_ptr() + guard
                b = a + nb + guard
                assert a % 16 == 0 and b % 16 == 0
                s = lbm.Simulation(*shape, q, name, w.tau, use_torch_memory=False)
                assert L.lbm_bind(s._h, a, b, torch.cuda.current_stream().cuda_stream) == 0
                s.set_variant(variant)
                s.set_flags(w.flags)
                s.init(w.rho, w.u)
                s.step(5)
                s.read_rho_u()
                s.close()
                torch.cuda.synchronize()
                canary = torch.cat([big[:guard], big[guard + nb:2 * guard + nb], big[2 * guard + 2 * nb:]])
                assert bool((canary == 0xA5).all()), (q, shape, name, variant)
