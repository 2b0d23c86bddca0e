"""-m gpu: md_kinetic_noalloc (kinetic energy and momentum with the block partials in the library's static __device__
array, no allocation) against the existing path, md_thermo on a context, within the tolerance test_thermo_reductions
uses (1e-12 of the kinetic energy, 1e-11 of sum |v| for the momentum), on two calls in a row that share the scratch
array.  Collected last on purpose (pytest -x): nothing runs after it."""
import numpy as np
import pytest

from paper_1412_3387_b200 import binding as B
from paper_1412_3387_b200 import inputs

pytestmark = pytest.mark.gpu


def _existing_path(wl, mass=None):
    """md_thermo of a context holding the same velocities (and masses): the reduction this entry point is a variant of."""
    md = B.MD(wl.box, wl.N, wl.rc, wl.r_buff)
    md.set_state(wl.pos, wl.vel, mass)
    md.build_cells()
    md.forces_bonds(0.0, 1.0)                     # md_thermo wants a current force (for the potential); no bonds: zero
    t = md.thermo()
    return t["kinetic"], np.asarray(t["momentum"], dtype=np.float64)


def _check(out, ke, mom, vel_abs_sum):
    assert abs(out[0] - ke) < 1e-12 * ke
    assert np.abs(out[1:] - mom).max() < 1e-11 * vel_abs_sum


def test_kinetic_noalloc_matches_md_thermo_on_two_calls_in_a_row():
    import torch
    big = inputs.lj_fcc(14, rc=2.5, r_buff=0.4, kT=1.3, jitter=0.05, pos_seed=21, vel_seed=22)     # N = 10,976: 3 blocks, ragged
    small = inputs.lj_fcc(6, rc=2.5, r_buff=0.4, kT=0.8, jitter=0.05, pos_seed=23, vel_seed=24)     # N = 864: 1 block
    rng = np.random.default_rng(25)
    m_small = rng.uniform(0.5, 3.0, size=small.N)
    ke_b, mom_b = _existing_path(big)
    ke_s, mom_s = _existing_path(small, m_small)
    # plain sums as a third opinion on the existing path itself
    assert abs(ke_b - 0.5 * np.sum(big.vel ** 2)) < 1e-12 * ke_b
    assert abs(ke_s - 0.5 * np.sum(m_small[:, None] * small.vel ** 2)) < 1e-12 * ke_s

    d_vb = torch.from_numpy(big.vel).cuda()
    d_vs = torch.from_numpy(small.vel).cuda()
    d_ms = torch.from_numpy(m_small).cuda()
    out_b = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    out_s = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    out_r = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    B.kinetic_noalloc(d_vb, None, out_b, stream=stream)            # first use on this device: takes the symbol address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # two calls in a row on one stream, no synchronisation between them; the second one is SMALLER, so the scratch still
    # holds the first call's partials of blocks 1 and 2 when it runs and must not read them
    B.kinetic_noalloc(d_vb, None, out_b, stream=stream)
    B.kinetic_noalloc(d_vs, d_ms, out_s, stream=stream)
    B.kinetic_noalloc(d_vb, None, out_r, stream=stream)            # and back: bit-reproducible
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                   # the calls took no device memory
    hb, hs, hr = out_b.cpu().numpy(), out_s.cpu().numpy(), out_r.cpu().numpy()
    _check(hb, ke_b, mom_b, np.abs(big.vel).sum())
    _check(hs, ke_s, mom_s, np.abs(m_small[:, None] * small.vel).sum())
    assert hb.tolist() == hr.tolist()
    # a prefix of the array (n given), the default stream, and the empty system
    B.kinetic_noalloc(d_vb, None, out_s, n=5000)
    torch.cuda.synchronize()
    assert abs(out_s[0].item() - 0.5 * np.sum(big.vel[:5000] ** 2)) < 1e-12 * ke_b
    B.kinetic_noalloc(d_vb, None, out_s, n=0)
    torch.cuda.synchronize()
    assert out_s.cpu().numpy().tolist() == [0.0, 0.0, 0.0, 0.0]


def test_kinetic_noalloc_rejects_what_it_cannot_hold():
    import torch
    v = torch.zeros((16, 3), dtype=torch.float64, device="cuda")
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    with pytest.raises(B.MDError, match="exceeds MD_NOALLOC_MAX_N = 33554432"):
        B.kinetic_noalloc(v, None, out, n=B.MD_NOALLOC_MAX_N + 1)  # rejected before anything is read
    with pytest.raises(B.MDError, match="DEVICE pointers"):
        B.kinetic_noalloc(np.zeros((16, 3)), None, out)
    with pytest.raises(B.MDError, match="required"):
        B.kinetic_noalloc(v, None, None)
    B.kinetic_noalloc(v, None, out)                                 # still usable after the failures
    torch.cuda.synchronize()
    assert out.cpu().numpy().tolist() == [0.0, 0.0, 0.0, 0.0]
