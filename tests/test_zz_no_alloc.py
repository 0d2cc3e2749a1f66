"""dpi_forward_noalloc -- the entry point for callers that cannot allocate device memory.

Who that is: an embedding operator running inside a serving runtime whose arena already holds the whole GPU (tables plus
the framework's pool), a request thread that cannot afford the driver locks / device-wide synchronisation of cudaMalloc and
cudaFree, or a stateless callback with nowhere to keep a plan handle. For them the library keeps the fused forward
kernel's working memory in a fixed ~2 MB array inside its own image (csrc/forward_noalloc.cu) instead of in a dpi_plan_t.

What is checked here, on a GPU: the block it writes equals the one the existing path (dpi_forward through a plan, fused
launch) writes -- same kernel, so bit for bit, which is inside every tolerance of tests/parity.py -- and both agree with the
oracle within those tolerances; on TWO CALLS IN A ROW that share the array, the second with a different shape and a
different batch, so anything the first call left behind (counters, look-back records, offsets) would show.
Without a GPU: the size limit is enforced on the host before any CUDA call.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity tests.
It must pass alone in a fresh process (first use of the array) and after the rest of the suite (array already touched by
nothing else, but the device full of other plans' state).
"""
import numpy as np
import pytest
import torch

from paper_2606_21101_b200 import binding, harness, workloads as W
from tests.parity import assert_outputs_match, oracle_reference


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_21101_b200 import build
    build.build()
    binding.load_library()


def test_noalloc_rejects_batches_beyond_the_builtin_array():
    """More bags than the built-in array has room for: refused on the host, with the limit in the message (no GPU needed)."""
    lib = binding.load_library()
    T, B = 8, binding.NOALLOC_MAX_BAGS // 8 + 1
    st = lib.dpi_forward_noalloc(T, 16, binding.DPI_F32, B, 16, 16, 16, None, 16, None)   # pointers are never touched
    assert st == 1   # DPI_ERR_INVALID_ARG
    msg = lib.dpi_last_error().decode()
    assert "DPI_NOALLOC_MAX_BAGS" in msg and str(binding.NOALLOC_MAX_BAGS) in msg
    # the limit itself passes the size check and fails later, on the row size, still before any CUDA call
    st = lib.dpi_forward_noalloc(T, 3, binding.DPI_F32, binding.NOALLOC_MAX_BAGS // 8, 16, 16, 16, None, 16, None)
    assert st == 2 and "multiple of 16" in lib.dpi_last_error().decode()


class _Problem:
    """One seeded batch on the device, the block the existing path writes for it, and the oracle's block."""

    def __init__(self, cfg, batch_seed):
        self.cfg = cfg
        rows = cfg.table_rows()
        self.host_tables = [W.full_table_storage(cfg, t, int(rows[t])) for t in range(cfg.T)]
        self.dt = harness.tables_from_host(cfg, self.host_tables)
        self.batch = W.make_batch(cfg, rows, batch_seed)
        self.pooling = cfg.pooling_modes()
        self.db = harness.upload_batch(self.batch)
        # existing path: a plan, dpi_forward forced onto its fused single launch
        plan = harness.make_plan(cfg, rows, max(self.batch.N, 1))
        plan.set_option(binding.OPT_FUSED, 1)
        self.want = harness.new_output(cfg, fill_nan=True)
        plan.forward(self.db.lengths, self.dt.ptrs, self.db.indices, self.want, pooling=self.pooling)
        torch.cuda.synchronize()
        plan.destroy()
        self.ref = oracle_reference(self.host_tables, cfg.dtype, cfg.B, self.batch.lengths, self.batch.indices, self.pooling)

    def launch(self):
        """dpi_forward_noalloc into a fresh NaN-filled block; asynchronous."""
        cfg = self.cfg
        got = harness.new_output(cfg, fill_nan=True)
        before = binding.launch_count()
        binding.forward_noalloc(cfg.T, cfg.D, W.DTYPE_CODE[cfg.dtype], cfg.B, self.db.lengths, self.dt.ptrs, self.db.indices, got,
                                pooling=self.pooling)
        assert binding.launch_count() - before == 2   # the reset of the shared words + the fused forward kernel
        return got

    def check(self, got):
        cfg = self.cfg
        bits = torch.int16 if got.element_size() == 2 else torch.int32
        assert np.array_equal(got.view(bits).cpu().numpy(), self.want.view(bits).cpu().numpy())   # same kernel: bit for bit
        assert_outputs_match(harness.out_to_f64(got), self.ref, self.batch.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out)


@pytest.mark.gpu
def test_noalloc_matches_the_plan_path_on_two_calls_in_a_row():
    harness.require_cuda()
    # a: c3-shaped (22 fp16 tables, bags of 1..3, mean pooling, Zipf ids), 45 056 bags = hundreds of chunks;
    # b: c1 (4 fp32 tables, 128 samples, sum) -- a handful of chunks and another dtype, so counters, look-back records or
    #    offsets left over from the call before would show;
    # c: long bf16 bags (Poisson(20), 5 % empty, half the tables mean-pooled: the warp-per-bag body)
    a = _Problem(W.Config("na3", 22, ("loguniform", 100, 5e4), 32, "f16", 2048, ("uniform", 1, 3), ("zipf", 1.2), "mean", 0), 11)
    b = _Problem(W.CONFIGS["c1"], 12)
    c = _Problem(W.Config("na4", 5, (1000, 17, 4000, 1, 250), 64, "bf16", 333, ("poisson", 20.0, 100, 0.05), ("zipf", 1.05), "half", 7), 13)
    # two calls in a row on one stream, nothing in between (no synchronisation, no other kernel): large then small
    got_a, got_b = a.launch(), b.launch()
    torch.cuda.synchronize()
    a.check(got_a)
    b.check(got_b)
    # and again the other way round, then the long-bag shape, then the first shape over a shorter call's leftovers
    outs = [(p, p.launch()) for p in (b, a, c, a)]
    torch.cuda.synchronize()
    for p, got in outs:
        p.check(got)


@pytest.mark.gpu
def test_noalloc_takes_a_batch_at_the_size_limit():
    """G = DPI_NOALLOC_MAX_BAGS exactly (one-hot, 8 tables): the last offset lands in the array's last word."""
    harness.require_cuda()
    T, D = 8, 16
    B = binding.NOALLOC_MAX_BAGS // T
    g = torch.Generator(device="cpu").manual_seed(5)
    rows = 1000
    tables = [torch.rand((rows, D), generator=g, dtype=torch.float32).cuda() for _ in range(T)]
    ptrs = torch.tensor([t.data_ptr() for t in tables], dtype=torch.int64, device="cuda")
    ids = torch.randint(0, rows, (B, T), generator=g, dtype=torch.int32)
    lengths = torch.ones(B * T, dtype=torch.int32, device="cuda")
    out = torch.full((B, T * D), float("nan"), dtype=torch.float32, device="cuda")
    for _ in range(2):
        out.fill_(float("nan"))
        binding.forward_noalloc(T, D, binding.DPI_F32, B, lengths, ptrs, ids.cuda().reshape(-1), out)
        torch.cuda.synchronize()
        want = torch.cat([tables[t][ids[:, t].long().cuda()] for t in range(T)], dim=1)   # a bag of length 1 is its row
        assert torch.equal(out, want)
