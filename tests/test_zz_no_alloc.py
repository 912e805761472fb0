"""nnp_coupling_compute_static: the Eq. 4 coupling term through the entry point that allocates nothing (its scratch is a
file-scope device array of a fixed maximum size) against the existing handle path (nnp_coupling_create +
nnp_coupling_compute), on two calls in a row that share the scratch array.  Collected last on purpose (file name)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle.coupling_oracle import COULOMB_KCAL_A  # noqa: E402
from paper_2201_08110_b200 import binding  # noqa: E402
from paper_2201_08110_b200 import workloads as wl  # noqa: E402
from paper_2201_08110_b200.binding import Coupling, NNPError  # noqa: E402

F_TOL = 1e-3  # kcal/mol/A (north_star), as in tests/test_gpu_extras.py
DEV = "cuda:0"


def _existing_path(s, cutoff, f0):
    """Energy and the force buffer after nnp_coupling_compute added into a copy of f0."""
    cp = Coupling(s.nnp_rows, s.q_nnp, s.sigma_nnp, s.eps_nnp, s.mm_rows, s.q_mm, s.sigma_mm, s.eps_mm,
                  coulomb_const=COULOMB_KCAL_A, cutoff=cutoff)
    pos = torch.from_numpy(s.positions).to(DEV)
    E = torch.full((1,), float("nan"), dtype=torch.float64, device=DEV)
    F = torch.from_numpy(f0.copy()).to(DEV)
    cp.compute(pos.data_ptr(), 3, E.data_ptr(), F.data_ptr(), 3, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    out = E.item(), F.cpu().numpy()
    cp.destroy()
    return out


def _device_inputs(s, f0):
    d = lambda a, t: torch.from_numpy(np.ascontiguousarray(a, dtype=t)).to(DEV)
    lists = [d(s.nnp_rows, np.int32), d(s.q_nnp, np.float32), d(s.sigma_nnp, np.float32), d(s.eps_nnp, np.float32),
             d(s.mm_rows, np.int32), d(s.q_mm, np.float32), d(s.sigma_mm, np.float32), d(s.eps_mm, np.float32)]
    pos = torch.from_numpy(s.positions).to(DEV)
    E = torch.full((1,), float("nan"), dtype=torch.float64, device=DEV)
    F = torch.from_numpy(f0.copy()).to(DEV)
    return lists, pos, E, F


def _static_call(s, cutoff, lists, pos, E, F):
    p = [t.data_ptr() for t in lists]
    binding.coupling_compute_static(len(s.nnp_rows), p[0], p[1], p[2], p[3], len(s.mm_rows), p[4], p[5], p[6], p[7],
                                    COULOMB_KCAL_A, cutoff, 1.0, pos.data_ptr(), 3, E.data_ptr(), F.data_ptr(), 3,
                                    torch.cuda.current_stream().cuda_stream)


def test_static_entry_point_matches_the_handle_path_on_two_calls_in_a_row():
    # a large system first, then a small one without cutoff: the second call finds the first call's partial sums and
    # atom records in the shared scratch array and must not be affected by them
    cases = [(wl.coupling_system(n_mm=30000, seed=wl.BASE_SEED + 91), 9.0),
             (wl.coupling_system(n_mm=700, seed=wl.BASE_SEED + 92), 0.0)]
    rng = np.random.default_rng(3)
    f0s = [rng.normal(size=(s.n_rows, 3)).astype(np.float32) for s, _ in cases]
    ref = [_existing_path(s, rc, f0) for (s, rc), f0 in zip(cases, f0s)]
    dev = [_device_inputs(s, f0) for (s, _), f0 in zip(cases, f0s)]  # all inputs and outputs exist before the calls
    binding.coupling_static_init()
    torch.cuda.synchronize()
    for (s, rc), d in zip(cases, dev):  # back to back on one stream, no synchronisation in between
        _static_call(s, rc, *d)
    torch.cuda.synchronize()
    for k, ((s, rc), d, (V, F)) in enumerate(zip(cases, dev, ref)):
        e, f = d[2].item(), d[3].cpu().numpy()
        fmax = np.abs(F - f0s[k]).max()
        print(f"[no-alloc] call {k}: n_mm={len(s.mm_rows)} cutoff={rc}: V={V:.6f} |dV|={abs(e - V):.2e} "
              f"max|dF|={np.abs(f - F).max():.2e} (max|F| {fmax:.1f}) identical={e == V and np.array_equal(f, F)}")
        assert np.isfinite(e) and fmax > 1.0
        assert abs(e - V) <= 1e-9 * max(1.0, abs(V))
        assert np.abs(f - F).max() <= max(F_TOL * 1e-2, 2e-7 * fmax)
    # a third call (the first system again, into a fresh buffer) leaves the amount of free device memory unchanged
    s, rc = cases[0]
    lists, pos, E, F = _device_inputs(s, f0s[0])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    _static_call(s, rc, lists, pos, E, F)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert abs(E.item() - ref[0][0]) <= 1e-9 * max(1.0, abs(ref[0][0]))
    assert np.abs(F.cpu().numpy() - ref[0][1]).max() <= max(F_TOL * 1e-2, 2e-7 * np.abs(ref[0][1] - f0s[0]).max())


def test_static_entry_point_rejects_sizes_beyond_its_scratch():
    for n_nnp, n_mm in ((binding.COUPLING_STATIC_MAX_NNP + 1, 10), (10, binding.COUPLING_STATIC_MAX_MM + 1)):
        with pytest.raises(NNPError) as err:
            binding.coupling_compute_static(n_nnp, None, None, None, None, n_mm, None, None, None, None, COULOMB_KCAL_A,
                                            9.0, 1.0, None, 3, None, None, 3, 0)
        assert err.value.code == -7 and "STATIC_LIMIT" in str(err.value)
