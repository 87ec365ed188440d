"""pt_energy_static (include/pt.h): the allocation-free entry point -- total energies of caller-supplied configurations
with the recount's scratch (coupling table, packed spins) in a file-scope device array -- against the existing path
(pt_create + pt_set_spins + pt_energy(recompute)) and against the oracle's O(L^2) recount.  Integer work: bit-exact.

This file is collected last on purpose (the suite runs with pytest -x): it must pass alone in a fresh process and
after all other tests."""
import numpy as np
import pytest

from paper_1308_5426_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pt():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test on a box without CUDA")
    from paper_1308_5426_b200 import build
    build.build()
    from paper_1308_5426_b200 import pt as ptmod
    return ptmod


def existing_path_energy(pt, L, q, sigma, spins):
    """E of the configurations spins[n_conf, L] through a context: set_spins, then the O(L^2) recount."""
    n_conf = spins.shape[0]
    g = pt.PT(L, q, sigma, 1, n_conf, np.linspace(0.5, 1.5, n_conf), 4242)
    g.set_spins(spins.reshape(1, n_conf, L))
    E = g.energy(recompute=True).reshape(n_conf).copy()
    g.close()
    return E


def static_energy(pt, L, q, sigma, spins, E_dev, status_dev):
    import torch
    s_dev = torch.from_numpy(np.ascontiguousarray(spins)).cuda()
    n_conf = spins.shape[0]
    pt.energy_static(L, q, sigma, s_dev, n_conf, E_dev, status_dev, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return E_dev[:n_conf].cpu().numpy().copy(), int(status_dev.item())


def test_static_energy_equals_existing_path_two_calls_in_a_row(pt, oracle):
    import torch
    E_dev = torch.full((256,), -7, dtype=torch.int64, device="cuda")
    status_dev = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    # two calls in a row on the shared scratch; the second is smaller in every way (L, q, n_conf, narrower packing),
    # so anything left over from the first call that it read would show
    shapes = [(1024, 37, 0.45, 24), (200, 5, 0.8, 3)]
    for (L, q, sigma, n_conf) in shapes:
        spins = inputs.random_spins(1, n_conf, L, q, seed=L + q).reshape(n_conf, L)
        got, status = static_energy(pt, L, q, sigma, spins, E_dev, status_dev)
        want = existing_path_energy(pt, L, q, sigma, spins)
        assert status == 0
        np.testing.assert_array_equal(got, want, err_msg="L=%d q=%d" % (L, q))
        o = oracle.Oracle(L, q, sigma, 1, n_conf, np.linspace(0.5, 1.5, n_conf), 1)
        o.set_spins(spins.reshape(1, n_conf, L))
        np.testing.assert_array_equal(got, o.energy(recompute=True).reshape(n_conf))
        o.close()
    # the first shape again: same result after the scratch held something else
    L, q, sigma, n_conf = shapes[0]
    spins = inputs.random_spins(1, n_conf, L, q, seed=L + q).reshape(n_conf, L)
    again, status = static_energy(pt, L, q, sigma, spins, E_dev, status_dev)
    np.testing.assert_array_equal(again, existing_path_energy(pt, L, q, sigma, spins))
    assert status == 0


def test_static_energy_headline_shape_and_ground_state(pt):
    """configs[3]'s shape (128 x 4096 sites: half the scratch), hot-start spins of the method; and the all-equal
    configuration, whose energy is -(L/2) sum_r Jq[r] (every pair counts)."""
    import torch
    w = inputs.config(3)
    g = pt.PT(w.L, w.q, w.sigma, 1, w.n_rep, inputs.betas(w), w.seed)
    spins = g.get_spins().reshape(w.n_rep, w.L)
    want = g.energy(recompute=True).reshape(w.n_rep).copy()
    Jq = g.get_couplings().astype(np.int64)
    g.close()
    E_dev = torch.zeros(w.n_rep, dtype=torch.int64, device="cuda")
    status_dev = torch.zeros(1, dtype=torch.int32, device="cuda")
    got, status = static_energy(pt, w.L, w.q, w.sigma, spins, E_dev, status_dev)
    assert status == 0
    np.testing.assert_array_equal(got, want)
    ones = np.full((2, w.L), 3, dtype=np.uint8)
    got, status = static_energy(pt, w.L, w.q, w.sigma, ones, E_dev, status_dev)
    assert status == 0
    assert got.tolist() == [-(w.L // 2) * int(Jq.sum())] * 2


def test_static_energy_limits_and_bad_colours(pt):
    import torch
    E_dev = torch.zeros(8, dtype=torch.int64, device="cuda")
    status_dev = torch.zeros(1, dtype=torch.int32, device="cuda")
    s_dev = torch.ones(64, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    for (L, q, sigma, n_conf) in [(pt.STATIC_MAX_L + 8, 3, 0.5, 1),            # L beyond the maximum
                                  (4096, 3, 0.5, pt.STATIC_MAX_SITES // 4096 + 1),  # n_conf * L beyond the maximum
                                  (60, 3, 0.5, 1), (64, 65, 0.5, 1), (64, 3, 0.0, 1), (64, 3, 0.5, 0)]:
        with pytest.raises(pt.PTError) as ei:
            pt.energy_static(L, q, sigma, s_dev, n_conf, E_dev, status_dev, stream)
        assert ei.value.code in (-1, -5)
        if L > pt.STATIC_MAX_L or n_conf * L > pt.STATIC_MAX_SITES:
            assert ei.value.code == -5 and "exceeds" in str(ei.value)
    # a colour outside 1..q is reported through status_dev, and the flag does not stick to the next call
    bad = np.ones((1, 64), dtype=np.uint8)
    bad[0, 17] = 4
    _, status = static_energy(pt, 64, 3, 0.5, bad, E_dev, status_dev)
    assert status == 1
    bad[0, 17] = 0
    _, status = static_energy(pt, 64, 3, 0.5, bad, E_dev, status_dev)
    assert status == 1
    good = np.ones((1, 64), dtype=np.uint8)
    _, status = static_energy(pt, 64, 3, 0.5, good, E_dev, status_dev)
    assert status == 0
    # status_dev may be NULL
    pt.energy_static(64, 3, 0.5, s_dev, 1, E_dev, None, stream)
    torch.cuda.synchronize()
