"""hqmc_action_boson_noalloc (include/hqmc.h): the allocation-free S_B entry point against the existing path
(hqmc_energies' S_B on a context), within the tolerance the energies parity test uses (1e-11 relative), on calls in a row
that share the library's static scratch.  Collected last on purpose (file name): the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2508_16298_b200 import inputs

TOL = 1e-11


def _existing_SB(hq, theta_dev, L, Nt, c_tau, K, compact):
    g = hq.HQMC(L, Nt, c_tau=c_tau, K=K, compact=compact, W=min(6, Nt - 1))
    g.set_theta(theta_dev)
    SB = g.energies()[0]
    g.close()
    return SB


@pytest.mark.gpu
def test_noalloc_matches_existing_path_on_calls_in_a_row(cuda_device):
    from paper_2508_16298_b200 import hqmc as hq
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    # a lattice of several CTAs with a ragged last one (2 * 18^2 * 7 = 4536 links), twice with different fields, then a
    # bigger one (config 3 size: 73 728 links = 18 partials) and a smaller one again: stale partials must not leak
    cases = [(18, 7, 3, 1.3, 0.7, True), (18, 7, 4, 1.3, 0.7, True), (24, 64, 5, 0.8, 1.1, False), (4, 8, 6, 1.3, 0.7, True),
             (6, 10, 7, 2.0, -0.5, False)]
    for L, Nt, seed, c_tau, K, compact in cases:
        theta = torch.from_numpy(inputs.theta_uniform(L, Nt, seed)).cuda()
        ref = _existing_SB(hq, theta, L, Nt, c_tau, K, compact)
        out.fill_(float("nan"))
        hq.action_boson_noalloc(theta, L, Nt, c_tau, K, compact, out)
        got1 = float(out[0].item())
        out1 = out[1:]
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        hq.action_boson_noalloc(theta, L, Nt, c_tau, K, compact, out1)          # second call in a row, same stream
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0                            # the call took no device memory
        got2 = float(out[1].item())
        assert abs(got1 - ref) <= TOL * abs(ref) + TOL, (L, Nt, got1, ref)
        assert got2 == got1, (L, Nt, got1, got2)                              # fixed partition: deterministic bit for bit


@pytest.mark.gpu
def test_noalloc_back_to_back_without_sync_and_on_a_side_stream(cuda_device):
    from paper_2508_16298_b200 import hqmc as hq
    L, Nt = 12, 14
    th = [torch.from_numpy(inputs.theta_uniform(L, Nt, s)).cuda() for s in (11, 12)]
    ref = [_existing_SB(hq, t, L, Nt, 1.3, 0.7, True) for t in th]
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):                                  # two calls enqueued back to back on ONE stream: ordered
        hq.action_boson_noalloc(th[0], L, Nt, 1.3, 0.7, True, out[0:])
        hq.action_boson_noalloc(th[1], L, Nt, 1.3, 0.7, True, out[1:])
    side.synchronize()
    got = out.cpu().numpy()
    assert np.all(np.abs(got - np.array(ref)) <= TOL * np.abs(ref) + TOL), (got, ref)


def test_noalloc_rejects_sizes_beyond_the_static_scratch():
    """Argument checks come before any CUDA call, so this runs without a GPU: 2 L^2 Ntau > 2^25 links -> HQMC_EINVAL + text."""
    from paper_2508_16298_b200 import hqmc as hq
    lib = C.CDLL(hq.LIB_PATH)
    lib.hqmc_last_error.restype = C.c_char_p
    fn = lib.hqmc_action_boson_noalloc
    fn.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_void_p, C.c_void_p]
    fake = C.c_void_p(4096)                                        # never dereferenced: the size check fails first
    assert hq.NOALLOC_MAX_LINKS == 1 << 25
    assert fn(fake, 4096, 2, 1.0, 1.0, 1, fake, None) == hq.HQMC_EINVAL          # 2 * 4096^2 * 2 = 2^26 links
    assert b"HQMC_NOALLOC_MAX_LINKS" in lib.hqmc_last_error()
    assert fn(fake, 128, 1025, 1.0, 1.0, 1, fake, None) == hq.HQMC_EINVAL         # one slice over the limit
    assert fn(None, 4, 8, 1.0, 1.0, 1, fake, None) == hq.HQMC_EINVAL
    assert fn(fake, 4, 8, 1.0, 1.0, 1, None, None) == hq.HQMC_EINVAL
    assert fn(fake, 1, 8, 1.0, 1.0, 1, fake, None) == hq.HQMC_EINVAL


@pytest.mark.gpu
def test_noalloc_at_the_maximum_size_closed_form(cuda_device):
    """Exactly HQMC_NOALLOC_MAX_LINKS links (all 8192 partials in use; beyond the contexts' L <= 96): a constant field has
    zero curl and zero time differences, so S_B = K L^2 Ntau (compact: c_tau (1 - cos 0) = 0)."""
    from paper_2508_16298_b200 import hqmc as hq
    L, Nt = 128, 1024
    assert 2 * L * L * Nt == hq.NOALLOC_MAX_LINKS
    theta = torch.full((Nt, 2, L, L), 0.25, dtype=torch.float64, device="cuda")
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    hq.action_boson_noalloc(theta, L, Nt, 1.3, 0.7, True, out)
    assert abs(float(out.item()) - 0.7 * L * L * Nt) <= 1e-12 * 0.7 * L * L * Nt
    with pytest.raises(hq.HqmcError, match="HQMC_NOALLOC_MAX_LINKS"):
        big = torch.empty((Nt + 1) * 2 * L * L, dtype=torch.float64, device="cuda")
        hq.action_boson_noalloc(big, L, Nt + 1, 1.3, 0.7, True, out)
