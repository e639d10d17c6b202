"""rbq_diag_gather (the row-gather experiment of SURVEY.md 7, hard part 5): all four copy modes -- cp.async and TMA
tile::gather4, separate and interleaved K / V -- must deliver exactly the requested rows: the 64-bit sum of all gathered
32-bit words against the same sum computed with torch indexing (integer work: bit-exact), ragged row counts included."""
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_rows,density", [(5000, 0.5), (70001, 0.37), (4096, 1.0), (300, 0.02)])
def test_diag_gather_checksums(rot128, n_rows, density):
    import torch
    from paper_2606_31519_b200 import binding as rb
    g = torch.Generator(device="cuda")
    g.manual_seed(n_rows)
    c = rb.RaBitQCache(1, 4, 1, 256, torch.from_numpy(rot128[0]))
    K = torch.randn(n_rows, 128, device="cuda", generator=g).to(torch.bfloat16)
    V = torch.randn(n_rows, 128, device="cuda", generator=g).to(torch.bfloat16)
    rows = torch.nonzero(torch.rand(n_rows, device="cuda", generator=g) < density).flatten().to(torch.int32)
    rows = rows[torch.randperm(rows.numel(), device="cuda", generator=g)]       # any order, not only ascending

    def words(t):
        return (t[rows.long()].contiguous().view(torch.int32).to(torch.int64) & 0xFFFFFFFF).sum()

    want = int((words(K) + words(V)).item())
    KV = torch.cat([K, V], dim=1).contiguous()
    for mode in (0, 1, 2, 3):
        cs = torch.zeros(1, dtype=torch.int64, device="cuda")
        rb.rbq_diag_gather(c.ctx, K if mode < 2 else KV, V if mode < 2 else None, rows, mode, cs)
        rb.rbq_diag_gather(c.ctx, K if mode < 2 else KV, V if mode < 2 else None, rows, mode, cs)   # the checksum accumulates
        torch.cuda.synchronize()
        assert int(cs.item()) == 2 * want, f"mode {mode}: gathered words differ"
    c.close()
