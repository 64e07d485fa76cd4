"""GPU test of the entry point that allocates nothing: mas_draft_entropy_static (include/msas.h; Eq. 9-10)
against the existing mas_draft_entropy, which takes its scratch from the caller.  Both run the same kernels, so the results are
compared bit for bit (which is inside the 2e-4 tolerance the oracle parity tests of this entry use), and against the oracle at
that tolerance.  Two calls in a row share the one static scratch array: the second must not see anything of the first.

In a file of its own that pytest collects last (the suite runs with `pytest -x`)."""
import numpy as np
import pytest
import torch

from oracle import mas_ref as O
from paper_2604_02945_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2604_02945_b200 import binding
    return binding


def _check_against_existing_path(B, n, V, dtype, seed, theta):
    L = synth.draft_logits(seed=seed, n_rows=n, V=V, dtype=dtype)
    dev = B.to_device(L)
    H_ref, sp_ref = B.draft_entropy(dev, theta)                      # the existing path: workspace from torch's allocator
    H = torch.full((n,), -7.0, dtype=torch.float32, device="cuda")   # outputs are the caller's: poisoned first
    sp = torch.full((n,), 9, dtype=torch.uint8, device="cuda")
    B.draft_entropy_static(dev, theta, H, sp)
    torch.cuda.synchronize()
    Hg, Hr = H.cpu().numpy(), H_ref.cpu().numpy()
    assert np.array_equal(Hg, Hr), np.abs(Hg.astype(np.float64) - Hr).max()
    assert np.array_equal(sp.cpu().numpy(), sp_ref.cpu().numpy())
    H_o, f_o = O.draft_entropy(L, theta)                             # and the oracle, at the tolerance of the parity tests
    assert np.all(np.abs(Hg.astype(np.float64) - H_o) <= 2e-4 * np.abs(H_o) + 2e-4)
    decided = np.abs(H_o - theta) > 1e-3
    assert np.array_equal(sp.cpu().numpy()[decided], f_o[decided])


def test_static_scratch_entry_matches_existing_path_on_two_calls_in_a_row(B):
    # a long-vocabulary call that splits every row over many CTAs (many partial triples), then a call of another shape and dtype
    # that reuses the head of the same scratch array, then the first shape again
    _check_against_existing_path(B, 16, 151936, "bf16", seed=21, theta=2.5)
    _check_against_existing_path(B, 700, 4100, "f32", seed=22, theta=2.0)
    _check_against_existing_path(B, 16, 151936, "bf16", seed=23, theta=2.5)


def test_static_scratch_entry_allocates_nothing_and_rejects_oversize(B):
    n, V = 64, 32000
    dev = B.to_device(synth.draft_logits(seed=31, n_rows=n, V=V, dtype="bf16"))
    H = torch.empty(n, dtype=torch.float32, device="cuda")
    sp = torch.empty(n, dtype=torch.uint8, device="cuda")
    B.draft_entropy_static(dev, 2.5, H, sp)                          # first call on this device: the symbol look-up
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    reserved0 = torch.cuda.memory_reserved()
    for _ in range(3):
        B.draft_entropy_static(dev, 2.5, H, sp)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0 and torch.cuda.memory_reserved() == reserved0
    # beyond the static array: one slice per row from 4 x SM count rows on, so n_rows > MAX_PARTIALS does not fit
    n_big = B.DRAFT_ENTROPY_STATIC_MAX_PARTIALS + 1
    big = torch.zeros((n_big, 8), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(B.MasError) as ei:
        B.draft_entropy_static(big, 2.5, torch.empty(n_big, dtype=torch.float32, device="cuda"), None)
    assert ei.value.status == B.MAS_ERR_WORKSPACE
    ok = torch.zeros((B.DRAFT_ENTROPY_STATIC_MAX_PARTIALS, 8), dtype=torch.bfloat16, device="cuda")   # the largest call that fits
    Hk = torch.empty(B.DRAFT_ENTROPY_STATIC_MAX_PARTIALS, dtype=torch.float32, device="cuda")
    B.draft_entropy_static(ok, 2.5, Hk, None)
    torch.cuda.synchronize()
    assert np.allclose(Hk.cpu().numpy(), np.log(8.0), atol=1e-5)     # uniform rows: H = ln V
