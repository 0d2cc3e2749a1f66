"""GPU parity (`-m gpu`) of dpi_forward_host -- the call behind bench.py's `e2e` number -- against the ORACLE, in the shapes the
round-2 review found untested: sample chunks (DPI_OPT_HOST_CHUNKS in {2, 7}: per-chunk sub-plans on three streams) together
with dpi_plan_set_columns (the block written into a wider row), with mixed per-table dims and with int64 ids. Chunks are
independent sub-batches, so every variant must give the block oracle.lookup_general defines (PAPER.md:143-164
generalised to bags; SURVEY.md 8(c) comparison rule). The full-size c4 / c5 runs of the same call are in test_gpu_parity.py
(`_every_sample_full_size`). Also here: int64 ids through the general kernel at an entry index >= 2^30 (the 64-bit shift of the
index address)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_21101_b200 import binding, harness, workloads as W
from tests.parity import assert_outputs_match_general, host_offsets

pytestmark = pytest.mark.gpu

ROWS = [1000, 17, 4000, 1, 250, 77]
POOL = np.asarray([0, 1, 0, 1, 1, 0], np.uint8)


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_21101_b200 import build
    build.build()
    binding.load_library()
    harness.require_cuda()


@pytest.mark.parametrize("chunks", [2, 7])
@pytest.mark.parametrize("direct_out", [1, 2])
@pytest.mark.parametrize("dims,dtype,out,idx64,custom_columns", [
    ([16, 16, 16, 16, 16, 16], "f32", "f32", False, True),      # set_columns only: equal dims, block inside a wider row
    ([16, 8, 32, 4, 64, 8], "f32", "f32", False, False),        # mixed dims only
    ([32, 8, 64, 16, 8, 40], "bf16", "f32", True, True),        # everything at once: mixed dims + columns + int64 ids + fp32 out
    ([32, 32, 32, 32, 32, 32], "f16", "f16", True, False),      # int64 ids only
])
def test_chunked_forward_host_with_the_interface_variants(dims, dtype, out, idx64, custom_columns, chunks, direct_out):
    T, B = len(dims), 333
    cfg = W.Config("fh", T, tuple(ROWS), max(dims), dtype, B, ("poisson", 4.0, 30, 0.1), ("zipf", 1.1), "sum", seed=21)
    batch = W.make_batch(cfg, np.asarray(ROWS, np.int64), 5)
    host_tables = W.mixed_dim_tables(cfg.seed, dims, ROWS, dtype)
    tables, ptrs = harness.tables_from_host_mixed(host_tables, dtype)
    ref = oracle.lookup_general(host_tables, W.DTYPE_CODE[dtype], B, batch.indices, host_offsets(batch.lengths).astype(np.int64), POOL)

    plan = binding.Plan(ROWS, np.asarray(dims, np.int32), W.DTYPE_CODE[dtype], B, max(batch.N, 1))
    if out != dtype:
        plan.set_out_dtype(W.DTYPE_CODE[out])
    if idx64:
        plan.set_layout(binding.BAGS_SAMPLE_MAJOR, binding.IDX_I64)
    elt = 4 if dtype == "f32" else 2
    dense_cols = np.concatenate(([0], np.cumsum(dims)[:-1])).astype(np.int64)
    cols = dense_cols
    if custom_columns:   # tables in reverse order with a 32-byte gap in front of each: a wider row, nothing at its dense place
        gap = 32 // elt
        cols = np.zeros(T, np.int64)
        c = 0
        for t in reversed(range(T)):
            c += gap
            cols[t] = c
            c += dims[t]
        plan.set_columns(cols)
    width = plan.plan_out_width()
    plan.set_option(binding.OPT_HOST_CHUNKS, chunks)
    plan.set_option(binding.OPT_HOST_DIRECT_OUT, direct_out)
    ln = torch.from_numpy(batch.lengths).pin_memory()
    idx = torch.from_numpy(batch.indices.astype(np.int64) if idx64 else batch.indices).pin_memory()
    out_host = torch.full((B, width), float("nan"), dtype=harness.TORCH_DTYPE[out]).pin_memory()
    for _ in range(2):   # the second call reuses the pipeline's sub-plans
        out_host.fill_(float("nan"))
        plan.forward_host(ptrs, ln, idx, out_host, pooling=POOL)
        got_wide = out_host.to(torch.float64).numpy()
        got = np.concatenate([got_wide[:, cols[t]:cols[t] + dims[t]] for t in range(T)], axis=1)   # back to the dense order
        assert_outputs_match_general(got, ref, batch.lengths.reshape(B, T), dims, dtype, out)
        if custom_columns and direct_out == 2:   # direct stores write the pooled vectors only: the gaps stay untouched (the staged
            # path copies whole rows of its device block back, so there the gaps hold unspecified values -- dpi.h says so)
            written = np.zeros(width, bool)
            for t in range(T):
                written[cols[t]:cols[t] + dims[t]] = True
            assert np.isnan(got_wide[:, ~written]).all()
    plan.destroy()


def test_int64_ids_through_the_general_kernel_beyond_2_pow_30_entries():
    """One batch whose index array holds 2^30 + 2^17 int64 ids (8.6 GB on the device, 32-bit offsets): the entry index of the
    last bags exceeds 2^30 and their byte offset 2^33, so the general kernel's `entry << idx_shift` has to be done in 64 bits
    (ADVICE r1). Same recipe as the 2^31-entry test of test_gpu_variants.py: 4098 bags of 262 176 entries over two tiny tables of
    16-byte rows whose values are multiples of 1/64, so sum pooling is exact in fp32 and compared bit for bit with the oracle."""
    free, _ = torch.cuda.mem_get_info()
    if free < 24 << 30:
        pytest.skip("needs 24 GB of free device memory")
    B, T, L = 2049, 2, 262176
    G = B * T
    N = G * L
    assert (1 << 30) < N < (1 << 31)
    rows = [1000, 37]
    rng = np.random.default_rng(8)
    lengths = np.full(G, L, np.int32)
    lengths[5] -= 3; lengths[6] += 3                                                   # not all equal
    block = rng.integers(0, 37, size=1 << 20).astype(np.int64)                         # valid for either table
    idx = np.tile(block, N // block.size + 1)[:N]
    tables = [(rng.integers(-8, 9, size=(r, 4)) / 64.0).astype(np.float32) for r in rows]   # sums stay exact in fp32
    off = np.concatenate(([0], np.cumsum(lengths.astype(np.int64))))
    plan = binding.Plan(rows, np.asarray([4, 4], np.int32), 0, B, N)
    plan.set_layout(binding.BAGS_SAMPLE_MAJOR, binding.IDX_I64)
    dev_tables, ptrs = harness.tables_from_host_mixed(tables, "f32")
    ln_dev = torch.from_numpy(lengths).cuda()
    idx_dev = torch.from_numpy(idx).cuda()
    pooling = np.array([0, 1], np.uint8)
    out = torch.full((B, 8), float("nan"), dtype=torch.float32, device="cuda")
    plan.build(ln_dev)
    assert plan.check_indices(idx_dev) == 0
    plan.lookup(ptrs, idx_dev, out, pooling=pooling)
    torch.cuda.synchronize()
    got = harness.out_to_f64(out)
    del idx_dev
    ref = oracle.lookup_general(tables, oracle.F32, B, idx, off, pooling)
    assert np.array_equal(got[:, :4], ref[:, :4])
    assert np.allclose(got[:, 4:], ref[:, 4:], rtol=1e-6, atol=1e-7)
    assert np.count_nonzero(off[:-1] >= (1 << 30)) >= 2   # whole bags past entry 2^30: the ones this test is about
    plan.destroy()
