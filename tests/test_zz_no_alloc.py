"""tkhp_polar_energy_static: the energy entry point for callers that cannot allocate.

Some users of libtkhp run where device allocation is off limits: a plug-in called inside an MD
engine's step loop once the engine's own pool owns all device memory, a callback that runs while
another thread has a stream capture open (the runtime refuses cudaMalloc then), a step loop that
cannot take cudaMalloc's device-wide stall.  They cannot give tkhp_create() a workspace, so they get
one call that works from a fixed 8,448-byte array inside the library's device image and takes only
their inputs and their output.  This file checks that call against the existing context path
(tkhp_polar_energy), which reduces in the same order, at the tolerance the energy tests of
tests/test_gpu_fullsize.py use (1e-12 relative), on calls made back to back: the array is shared and
keeps the previous call's partial sums and ticket, so a second call with other data and another grid
size is what would show stale scratch.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must
not hide the parity tests.  It passes alone in a fresh process (the first call does the per-device
address look-up) and after the other tests.
"""
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
COULOMB = 332.063713      # kcal A / (mol e^2), DESIGN.md U
REL_TOL = 1e-12           # as tests/test_gpu_fullsize.py: energy against a host FP64 evaluation


def test_entry_point_source_never_allocates():
    """The promise is static: the file that holds the entry point names no allocating call."""
    src = (ROOT / "paper_2011_01207_b200" / "csrc" / "energy_static.cu").read_text()
    code = re.sub(r"//[^\n]*", "", src)                  # the comments do name them
    for word in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMallocAsync", "cudaMallocManaged",
                 "cudaMemPool", "cudaHostRegister", "cudaStreamCreate", "cudaEventCreate", " new ", "malloc("):
        assert word not in code, word
    assert "static __device__ __align__(256) unsigned char g_energy_scratch" in code
    assert "cudaGetSymbolAddress" in code


def _host_energy(mu, field):
    return -0.5 * COULOMB * float(np.sum(mu.astype(np.float64) * field))


@pytest.mark.gpu
def test_static_energy_matches_context_path_on_consecutive_calls():
    import torch
    import paper_2011_01207_b200 as pk

    dev = torch.device("cuda", 0)
    rng = np.random.default_rng(20111207)
    # sizes: one CTA; a ragged tail; the headline system (grid capped at 1,024 CTAs, several strides);
    # then small again, so that the second-to-last call leaves 1,024 stale partials behind
    sizes = [1, 33, 98_304, 1_066_629, 700, 98_304]
    out = torch.full((len(sizes),), float("nan"), dtype=torch.float64, device=dev)
    expected_ctx, expected_host, cases = [], [], []
    for n in sizes:
        mu = rng.standard_normal((n, 3)) * 0.05
        field = rng.standard_normal((n, 3)) * 0.1
        mu_d, field_d = torch.as_tensor(mu, device=dev), torch.as_tensor(field, device=dev)
        cases.append((n, mu_d, field_d))
        expected_host.append(_host_energy(mu, field))
        # the existing path: a context (TILES mode needs no list for the energy), its workspace partials
        P = pk.Polarizer(n, box=0.0, precision=pk.TKHP_MIXED, list_mode=pk.TKHP_LIST_TILES)
        expected_ctx.append(float(P.polar_energy(mu_d, field_d).cpu()))
        P.close()
    # back-to-back calls on one stream, no synchronisation and nothing else in between
    stream = torch.cuda.current_stream(dev)
    for k, (n, mu_d, field_d) in enumerate(cases):
        pk.tkhp_polar_energy_static(0, n, mu_d, field_d, out[k:k + 1], stream)
    got = out.cpu().numpy()
    for k, n in enumerate(sizes):
        assert np.isfinite(got[k]), (n, got[k])
        assert abs(got[k] - expected_ctx[k]) <= REL_TOL * abs(expected_ctx[k]), (n, got[k], expected_ctx[k])
        assert abs(got[k] - expected_host[k]) <= REL_TOL * max(abs(expected_host[k]), 1e-3 * np.sqrt(n)), \
            (n, got[k], expected_host[k])
    # same inputs, same order of summation: the two calls on the 98,304-atom arrays differ only in which
    # stale scratch they found, and both equal the context path exactly
    n, mu_d, field_d = cases[2]
    pk.tkhp_polar_energy_static(0, n, mu_d, field_d, out[0:1], stream)
    pk.tkhp_polar_energy_static(0, n, mu_d, field_d, out[1:2], stream)
    again = out[:2].cpu().numpy()
    assert again[0] == again[1] == got[2] == expected_ctx[2]


@pytest.mark.gpu
def test_static_energy_rejects_what_it_cannot_hold():
    import torch
    import paper_2011_01207_b200 as pk

    dev = torch.device("cuda", 0)
    a = torch.ones(3, dtype=torch.float64, device=dev)
    e = torch.full((1,), 7.0, dtype=torch.float64, device=dev)
    with pytest.raises(pk.TkhpError) as too_big:      # only the count is looked at: nothing is launched
        pk.tkhp_polar_energy_static(0, pk.TKHP_STATIC_MAX_ATOMS + 1, a, a, e)
    assert too_big.value.code == pk.binding.TKHP_ECAPACITY and "TKHP_STATIC_MAX_ATOMS" in str(too_big.value)
    with pytest.raises(pk.TkhpError) as empty:
        pk.tkhp_polar_energy_static(0, 0, a, a, e)
    assert empty.value.code == pk.binding.TKHP_EINVAL
    with pytest.raises(pk.TkhpError) as null:
        pk.tkhp_polar_energy_static(0, 1, a, None, e)
    assert null.value.code == pk.binding.TKHP_EINVAL
    with pytest.raises(pk.TkhpError) as bad_dev:
        pk.tkhp_polar_energy_static(64, 1, a, a, e, stream=0)
    assert bad_dev.value.code == pk.binding.TKHP_EINVAL
    torch.cuda.synchronize(dev)
    assert float(e.cpu()) == 7.0                       # a refused call leaves the output alone
    pk.tkhp_polar_energy_static(0, 1, a, a, e)         # and the entry point still works afterwards
    assert abs(float(e.cpu()) + 1.5 * COULOMB) <= REL_TOL * 1.5 * COULOMB
