"""-m gpu: ocgs_staging_probe (diagnostic): each of the three staging methods -- __ldg, cp.async, TMA tile::gather4 -- must bring the
rows the rank list names into shared memory; the per-thread sums the kernels write are compared with the same sums by numpy."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _expected(rec, ranks, blocks, iters, batch):
    n = len(ranks)
    tid = np.arange(256)
    out = np.zeros((blocks, 256), np.float64)
    for b in range(blocks):
        for it in range(iters):
            base = ((b * iters + it) * batch) % n
            for k in range(batch // 32):
                e = (tid + 32 * k) & (batch - 1)
                rows = ranks[(base + e) % n]
                part = tid % 6
                vals = rec[rows[:, None], (4 * part)[:, None] + np.arange(4)[None, :]]
                out[b] += vals.astype(np.float64).sum(1)
    return out


def test_three_staging_methods_gather_the_right_rows():
    import torch
    from paper_2501_08174_b200 import binding as B
    rng = np.random.default_rng(3)
    n_rec, n_ranks, iters = 5000, 4096 + 37, 3
    rec = rng.uniform(-1, 1, (n_rec, 24)).astype(np.float32)
    ranks = rng.integers(0, n_rec, n_ranks).astype(np.uint32)
    rec_t = torch.tensor(rec, device="cuda"); ranks_t = torch.tensor(ranks.view(np.int32), device="cuda")
    blocks = torch.cuda.get_device_properties(0).multi_processor_count * 6
    for kind, batch in ((0, 256), (1, 128), (2, 128)):
        out = torch.zeros(blocks * 256, device="cuda")
        try:
            nbytes = B.ocgs_staging_probe(kind, rec_t, ranks_t, n_rec, n_ranks, iters, out)
        except B.OcgsError as e:
            if kind == 2 and e.code == B.OCGS_ERR_UNSUPPORTED:
                pytest.skip("driver without cuTensorMapEncodeTiled")
            raise
        torch.cuda.synchronize()
        assert nbytes == blocks * iters * batch * 96
        got = out.cpu().numpy().reshape(blocks, 256)
        exp = _expected(rec, ranks, 8, iters, batch)  # the first 8 CTAs are enough (every CTA runs the same code)
        assert np.allclose(got[:8], exp, rtol=0, atol=2e-4), kind
        assert np.abs(got).max() > 1.0
