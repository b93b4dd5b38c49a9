"""-m gpu: ocgs_masked_l1_static -- the entry point that allocates nothing (scratch in a static device array of the library) --
against the existing ocgs_masked_l1 path (scratch in the caller's workspace), on two calls in a row.

Collected last on purpose (the suite runs with pytest -x: a failure here must not hide other tests); passes alone in a fresh
process and after the other tests (the static array keeps whatever the last call left in it; no call reads a slot it has not
written)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _both_paths(B, torch, W, H, seed, with_mask):
    rng = np.random.default_rng(seed)
    color = torch.tensor(rng.uniform(0, 1, (3, H, W)).astype(np.float32), device="cuda")
    target = torch.tensor(rng.uniform(0, 1, (3, H, W)).astype(np.float32), device="cuda")
    target[:, : H // 3] = color[:, : H // 3]  # a region of exact zeros of R - I (gradient 0 there)
    mask = torch.tensor((rng.uniform(size=(H, W)) < 0.6).astype(np.uint8), device="cuda") if with_mask else None
    # existing path: partial sums in the caller's workspace
    ws = B.alloc_workspace(1, W, H, 16)
    g_ref = torch.full((3, H, W), 7.0, device="cuda"); l_ref = torch.full((1,), 7.0, device="cuda")
    B.ocgs_masked_l1(color, target, mask, W, H, g_ref, l_ref, ws, 1, 16)
    # new path: no workspace; the torch allocator must not move either (the call takes pointers only)
    g_new = torch.full((3, H, W), -7.0, device="cuda"); l_new = torch.full((1,), -7.0, device="cuda")
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    B.ocgs_masked_l1_static(color, target, mask, W, H, g_new, l_new)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    # by definition (S20): loss = sum |M (R - I)| / (3HW), gradient = M sign(R - I) / (3HW)
    d = (color.double() - target.double()).cpu().numpy() * (1.0 if mask is None else (mask.cpu().numpy()[None] > 0))
    assert abs(float(l_new.item()) - np.abs(d).sum() / (3.0 * H * W)) < 1e-6
    return g_ref.cpu().numpy(), float(l_ref.item()), g_new.cpu().numpy(), float(l_new.item())


def test_masked_l1_static_matches_the_workspace_path_on_two_calls_in_a_row():
    import torch
    from paper_2501_08174_b200 import binding as B
    # call 1: the headline image size (7 500 partial sums); call 2: a small ragged image (28 partial sums) -- the array then still
    # holds 7 472 stale sums of call 1, none of which may be read; call 3: large again
    for W, H, seed, with_mask in ((1600, 1200, 1, True), (100, 70, 2, False), (1920, 1080, 3, True)):
        g_ref, l_ref, g_new, l_new = _both_paths(B, torch, W, H, seed, with_mask)
        assert np.array_equal(g_new, g_ref), (W, H)                  # dL/dcolor: bit-identical
        assert abs(l_new - l_ref) <= 1e-7, (W, H, l_new, l_ref)      # the tolerance test_gpu_parity.py uses for the L1 scalar
        assert l_new > 0.05 and (g_new == 0).any() and (g_new != 0).any()


def test_masked_l1_static_rejects_sizes_beyond_its_scratch():
    import torch
    from paper_2501_08174_b200 import binding as B
    assert B.OCGS_MASKED_L1_STATIC_MAX_PIXELS == 8192 * 256
    W, H = 2048, 1025  # one row more than the limit
    x = torch.zeros((3, H, W), device="cuda"); g = torch.full((3, H, W), 5.0, device="cuda"); loss = torch.full((1,), 5.0, device="cuda")
    with pytest.raises(B.OcgsError) as e:
        B.ocgs_masked_l1_static(x, x, None, W, H, g, loss)
    assert e.value.code == B.OCGS_ERR_CAPACITY and "at most 2097152" in str(e.value)
    torch.cuda.synchronize()
    assert float(loss.item()) == 5.0 and float(g.min().item()) == 5.0  # nothing was launched
    B.ocgs_masked_l1_static(x[:, :1024].contiguous(), x[:, :1024].contiguous(), None, W, 1024, g[:, :1024].contiguous(), loss)  # exactly the limit
    torch.cuda.synchronize()
    assert float(loss.item()) == 0.0
    with pytest.raises(B.OcgsError):
        B.ocgs_masked_l1_static(x, x, None, 0, H, g, loss)
