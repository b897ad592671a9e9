"""bh_direct_forces (Eq.2: the binary64 direct-sum reference on the GPU) against the oracle's direct sum,
and the acceleration-error experiment built on it (section 4.2.1)."""
import numpy as np
import pytest

import bh_inputs
import oracle

pytestmark = pytest.mark.gpu

# both sides sum ~n binary64 terms in different orders from the same fp32 inputs: relative difference ~ sqrt(n) ulp
REL_TOL = 1e-11


def _to_gpu(pm):
    import torch
    return torch.from_numpy(np.ascontiguousarray(pm)).cuda()


@pytest.mark.parametrize("n,eps", [(1, 0.01), (2, 0.0), (127, 0.01), (128, 0.0), (129, 0.05), (3000, 0.0), (3000, 0.01)])
def test_direct_forces_match_the_oracle(n, eps):
    from paper_1106_1900_b200 import direct_forces
    pm, _, _ = bh_inputs.make("c1", n=n, seed=23)
    got = direct_forces(_to_gpu(pm), eps).cpu().numpy()
    ref = oracle.direct(pm, eps)
    assert np.all(np.isfinite(got))
    if n == 1:
        assert np.all(got == 0.0) and np.all(ref == 0.0)
        return
    da = np.linalg.norm(got[:, :3] - ref[:, :3], axis=1) / np.linalg.norm(ref[:, :3], axis=1)
    dp = np.abs(got[:, 3] - ref[:, 3]) / np.abs(ref[:, 3])
    assert da.max() < REL_TOL and dp.max() < REL_TOL, (da.max(), dp.max())


def test_direct_forces_target_range_and_arguments():
    import torch
    from paper_1106_1900_b200 import BhError, direct_forces
    pm, _, _ = bh_inputs.make("c1", n=1000, seed=29)
    d = _to_gpu(pm)
    part = direct_forces(d, 0.01, 300, 431).cpu().numpy()
    ref = oracle.direct(pm, 0.01, 300, 431)
    assert np.all(np.isnan(part[:300])) and np.all(np.isnan(part[431:]))       # rows outside the range are not touched
    assert np.allclose(part[300:431], ref[300:431], rtol=REL_TOL, atol=0.0)
    for bad in [(0, 0), (5, 5), (-1, 10), (0, 1001), (10, 5)]:
        with pytest.raises(BhError):
            direct_forces(d, 0.01, *bad)
    with pytest.raises(BhError):
        direct_forces(d, -1.0)
    with pytest.raises(BhError):
        direct_forces(torch.from_numpy(pm), 0.01)                               # host memory is refused, not dereferenced


def test_momentum_conservation_of_the_direct_sum():
    """sum m a = 0 to rounding (P11)."""
    from paper_1106_1900_b200 import direct_forces
    pm, _, _ = bh_inputs.make("c1", n=4096, seed=31)
    a = direct_forces(_to_gpu(pm), 0.01).cpu().numpy()
    m = pm[:, 3].astype(np.float64)
    net = np.abs((m[:, None] * a[:, :3]).sum(axis=0)).max()
    assert net < 1e-13 * np.abs(m[:, None] * a[:, :3]).sum()


def test_acceleration_error_experiment():
    """Eq.2 on a small Plummer sphere: the tree error against the GPU direct sum equals the one against the oracle's direct
    sum, falls with theta, and at theta -> 0 only fp32 rounding is left."""
    from paper_1106_1900_b200 import accuracy
    rows = accuracy.run(8192, [0.8, 0.5, 0.3, 1e-3], 0.0, seed=37)
    med = [r["exceeded_by_50pct"] for r in rows]
    p1 = [r["exceeded_by_1pct"] for r in rows]
    assert med[0] > med[1] > med[2] > med[3] and p1[0] > p1[1] > p1[2] > p1[3]
    assert med[3] < 1e-6 and p1[3] < 1e-5                     # theta -> 0: every cell opened, the direct sum in fp32
    assert 1e-5 < med[1] < 1e-2                               # theta = 0.5 with quadrupoles
    assert all(r["exceeded_by_50pct"] <= r["exceeded_by_10pct"] <= r["exceeded_by_1pct"] <= r["max"] for r in rows)
    # the same experiment against the oracle's binary64 direct sum of the same (sorted) particles
    import torch  # noqa: F401
    from paper_1106_1900_b200 import BarnesHut
    pm, vel, _ = bh_inputs.make("c2", n=8192, seed=37)
    bh = BarnesHut(8192)
    bh.set_particles(pm, vel); bh.tree_build(); bh.compute_forces(0.5, 0.0)
    t = bh.export_tree()
    ps = oracle.tree_build(pm, vel).pos                     # the oracle's own sorted particles (the GPU's, bit for bit)
    assert np.array_equal(t["pos_mass"].cpu().numpy(), ps)
    err = accuracy.relative_error(t["acc_pot"].cpu().numpy(), oracle.direct(ps, 0.0))
    assert abs(accuracy.exceeded_by(err, 0.5) - med[1]) < 1e-6 * med[1] + 1e-12


def test_fp32_probes_report_sane_rates():
    import torch
    """bh_probe_fp32 (SURVEY.md 8(d)): every kind runs, is positive and below the nominal FP32 peak; argument errors."""
    import ctypes as C
    import __graft_entry__ as g
    g.build()
    from paper_1106_1900_b200 import load_library, probe_fp32
    p = probe_fp32()
    props = torch.cuda.get_device_properties(0)
    nominal = props.multi_processor_count * 128 * 2 * 2.1e9 / 1e12      # generous clock bound
    assert set(p) == {"ffma", "ffma2", "ffma2_shared_operand", "ffma2_broadcast_scalar", "pc_body", "pc_body_executed", "pp_body", "pp_body_executed"}
    for k, v in p.items():
        assert 1.0 < v < nominal, (k, v)
    assert p["pc_body_executed"] < p["pc_body"] and abs(p["pc_body_executed"] / p["pc_body"] - 56 / 64) < 1e-9
    lib = load_library()
    x = C.c_double()
    s = torch.empty(16, dtype=torch.float32, device="cuda")
    assert lib.bh_probe_fp32(0, s.data_ptr(), 64, C.byref(x), None) == -2          # scratch too small
    assert lib.bh_probe_fp32(9, s.data_ptr(), 64, C.byref(x), None) == -1
