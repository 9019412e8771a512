"""gm_kinetic_static -- the entry point that allocates nothing (per-block partial sums in a file-scope __device__ array of
libgm.so instead of the caller's workspace) -- against the existing path, gm_energies (k_energy: the same fp32 inputs, fp64
terms and sums), on calls in a row that share the array.  Tolerance: 1e-6 relative on the kinetic energy, as in the other
GPU tests; both sides differ in the order of the fp64 additions only.  Collected last on purpose (the suite runs with
pytest -x)."""
import numpy as np
import pytest

from workloads import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gm():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1310_2041_b200 import gm as g
    g.lib()
    return g


def existing_path(gm, w):
    s = gm.System(w)
    e = s.energies()
    s.close()
    return e["ke"], e["p"]


def static_path(gm, w, out):
    import torch
    vel = torch.from_numpy(np.ascontiguousarray(w.vel, np.float32)).cuda()
    mass = torch.from_numpy(np.ascontiguousarray(w.mass, np.float32)).cuda()
    gm.gm_kinetic_static(vel, mass, out)
    torch.cuda.synchronize()
    return out.cpu().numpy().copy()


def test_two_calls_in_a_row_match_gm_energies(gm):
    import torch
    wa = make_config("C3", scale=0.3)           # 27 000 beads: 27 CTAs, the last one ragged
    wb = make_config("C1")                      # 2 000 beads: 2 CTAs -- fewer than the call before left in the array
    rng = np.random.default_rng(5)
    wb.mass = rng.uniform(0.5, 2.0, wb.n).astype(np.float32)
    out = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    results = []
    for w in (wa, wb, wa):
        ke, p = existing_path(gm, w)
        r = static_path(gm, w, out)
        assert r[0] == pytest.approx(ke, rel=1e-6)
        scale = float(np.abs(w.mass[:, None] * w.vel).sum())
        assert np.abs(r[1:4] - p).max() <= 1e-9 * scale
        results.append(r)
    np.testing.assert_array_equal(results[0], results[2])          # nothing of the call in between leaks: bit-identical


def test_mass_defaults_to_one_and_empty_input(gm):
    import torch
    w = make_config("C1")
    vel = torch.from_numpy(w.vel).cuda()
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    gm.gm_kinetic_static(vel, None, out)
    torch.cuda.synchronize()
    v = w.vel.astype(np.float64)
    assert out[0].item() == pytest.approx(0.5 * (v * v).sum(), rel=1e-12)
    gm.gm_kinetic_static(vel[:0], None, out)
    torch.cuda.synchronize()
    assert (out.cpu().numpy() == 0.0).all()


def test_sizes_beyond_the_static_array_are_rejected(gm):
    import torch
    vel = torch.zeros((8, 3), dtype=torch.float32, device="cuda")
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    buf = gm.C.create_string_buffer(256)
    r = gm.lib().gm_kinetic_static(vel.data_ptr(), None, gm.GM_STATIC_MAX_BEADS + 1, 0, None, out.data_ptr(), buf, 256)
    assert r == gm.GM_ERR_INVALID_ARG and b"exceeds the static scratch array" in buf.value and b"8388608" in buf.value
    r = gm.lib().gm_kinetic_static(None, None, 8, 0, None, out.data_ptr(), buf, 256)
    assert r == gm.GM_ERR_INVALID_ARG


def test_capturable_in_a_cuda_graph(gm):
    # the use case the entry point exists for: one memset node + one kernel node, no allocation while capturing
    import torch
    w = make_config("C1")
    vel = torch.from_numpy(w.vel).cuda()
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    gm.gm_kinetic_static(vel, None, out)                    # outside the capture: resolves the array's address on this device
    torch.cuda.synchronize()
    expect = out.clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        gm.gm_kinetic_static(vel, None, out)
    for scale in (2.0, 3.0):
        vel.mul_(scale)
        expect = expect * torch.tensor([scale * scale, scale, scale, scale], dtype=torch.float64, device="cuda")
        out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert out[0].item() == pytest.approx(expect[0].item(), rel=1e-6)
        assert torch.allclose(out[1:], expect[1:], rtol=0, atol=1e-6 * float(np.abs(w.vel).sum()) * 6)
