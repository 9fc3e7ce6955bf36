"""hsma_direct_sum_static (include/hsma.h): the raw direct sum of Eq.(5) PAPER.md:64 for callers that cannot allocate
device memory -- every scratch buffer carved from one fixed 16 MiB `static __device__` array inside the library -- against
the existing path hsma_direct_sum (which cudaMallocs its scratch) and the oracle, on two calls in a row that share the
array.  Collected last on purpose (the file name): the suite runs with pytest -x.  All `-m gpu`."""
import numpy as np
import pytest

import hsma_workloads as W
from oracle import hsma_oracle as O

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_1806_04801_b200 as H
    H.binding.load_library()
    return H


def dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device="cuda")


def rel_inf(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def problem(seed, N, T, kind, L, shell, gamma):
    rng = np.random.default_rng(seed)
    Lh = np.asarray(L)
    src = (rng.random((N, 3)) - 0.5) * Lh
    q = rng.standard_normal(N)
    tgt = (rng.random((T, 3)) - 0.5) * Lh * 1.2
    return src, q, tgt, O.cell_table(kind, L, shell, gamma)


@pytest.mark.parametrize("refine", [1, 2])
def test_two_calls_in_a_row_match_the_allocating_path(H, refine):
    """Two different problems back to back on one stream, no synchronisation in between: the second call reuses (and
    overwrites) the scratch of the first -- a larger problem first, so stale contents lie behind the second one's buffers.
    Same kernels and launch shapes as hsma_direct_sum, so the results are equal bit for bit; the oracle at the bar the
    raw-kernel tests use (1e-12 of max|phi|)."""
    import torch
    cases = [problem(11, 5000, 3001, W.BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0),
             problem(12, 777, 1300, W.BC_MIRROR_CAVITY, (1.0, 1.2, 0.9), (1, 1, 1), -1.0)]
    args = [(dev(t), dev(s), dev(q), c) for s, q, t, c in cases]
    outs = [torch.empty(a[0].shape[0], dtype=torch.float64, device="cuda") for a in args]
    H.hsma_static_scratch_setup()
    t, s, q, c = args[1]                                           # (loads the kernels: module loading may allocate)
    H.hsma_direct_sum_static(t, s, q, c.shift, c.sign, c.w, c.central, -1, refine, outs[1])
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for (t, s, q, c), out in zip(args, outs):                      # two calls in a row, asynchronous
        H.hsma_direct_sum_static(t, s, q, c.shift, c.sign, c.w, c.central, -1, refine, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before             # no device memory was taken by the calls
    for (t, s, q, c), out, (src, qq, tgt, cells) in zip(args, outs, cases):
        old = torch.empty_like(out)
        H.hsma_direct_sum(t, s, q, c.shift, c.sign, c.w, c.central, -1, refine, old)
        assert torch.equal(out, old)
        assert rel_inf(out.cpu().numpy(), O.near_sum(tgt, src, qq, cells)) < 1e-12
    # and once more, the first problem again after the second has used the array
    t, s, q, c = args[0]
    again = torch.empty_like(outs[0])
    H.hsma_direct_sum_static(t, s, q, c.shift, c.sign, c.w, c.central, -1, refine, again)
    torch.cuda.synchronize()
    assert torch.equal(again, outs[0])


def test_self_exclusion_and_uniform_charges(H):
    """Targets are sources (bare self term skipped in the central cell only) with charges of equal magnitude: the
    uniform-|q| twin of the kernel is the one that runs, selected on the device from statistics kept in the scratch."""
    import torch
    N, t0, T = 4100, 700, 2055
    rng = np.random.default_rng(3)
    src = rng.random((N, 3)) - 0.5
    q = W.alternating_charges(N)
    cells = O.cell_table(W.BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0)
    ref = O.near_sum(src[t0:t0 + T], src, q, cells, self_offset=t0)
    for _ in range(2):
        out = torch.empty(T, dtype=torch.float64, device="cuda")
        H.hsma_direct_sum_static(dev(src[t0:t0 + T]), dev(src), dev(q), cells.shift, cells.sign, cells.w, cells.central,
                                 t0, 1, out)
        torch.cuda.synchronize()
        old = torch.empty_like(out)
        H.hsma_direct_sum(dev(src[t0:t0 + T]), dev(src), dev(q), cells.shift, cells.sign, cells.w, cells.central, t0, 1, old)
        assert torch.equal(out, old)
        assert rel_inf(out.cpu().numpy(), ref) < 1e-12


@pytest.mark.parametrize("byte", [0xFF, 0x00, 0x7F])
def test_reads_nothing_left_behind_in_the_scratch(H, byte):
    """The array keeps whatever the last call (or the fill hook) left: poisoned with NaN bytes, zeros or large finite
    garbage, the next call still equals the allocating path bit for bit -- every scratch word it reads, it wrote."""
    import torch
    for seed, N, T in ((21, 2311, 77), (22, 256, 4000)):
        src, q, tgt, c = problem(seed, N, T, W.BC_SLAB_XY_PERIODIC_Z_MIRROR, (1.0, 1.0, 0.5), (1, 1, 1), 0.5)
        t, s_, q_ = dev(tgt), dev(src), dev(q)
        out, old = torch.empty(T, dtype=torch.float64, device="cuda"), torch.empty(T, dtype=torch.float64, device="cuda")
        H.hsma_static_scratch_fill(byte)
        H.hsma_direct_sum_static(t, s_, q_, c.shift, c.sign, c.w, c.central, -1, 2, out)
        torch.cuda.synchronize()
        H.hsma_direct_sum(t, s_, q_, c.shift, c.sign, c.w, c.central, -1, 2, old)
        assert torch.equal(out, old) and bool(torch.isfinite(out).all())
        assert rel_inf(out.cpu().numpy(), O.near_sum(tgt, src, q, c)) < 1e-12


def test_limits_are_rejected_with_a_clear_error(H):
    """N, T > 65,536 or C > 32: HSMA_ERR_TOO_LARGE, nothing launched, output untouched; the maximum itself runs."""
    import torch
    assert H.hsma_static_scratch_bytes() == 16 << 20
    cells = O.cell_table(W.BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0)
    big = O.cell_table(W.BC_SLAB_XY_PERIODIC_Z_MIRROR, (1.0, 1.0, 0.5), (1, 1, 2), 0.5)      # 45 cells > 32
    rng = np.random.default_rng(4)

    def call(N, T, c):
        src, q, tgt = dev(rng.random((N, 3)) - 0.5), dev(rng.standard_normal(N)), dev(rng.random((T, 3)) - 0.5)
        out = torch.full((T,), -7.0, dtype=torch.float64, device="cuda")
        H.hsma_direct_sum_static(tgt, src, q, c.shift, c.sign, c.w, c.central, -1, 1, out)
        torch.cuda.synchronize()
        return src, q, tgt, out

    launches = H.hsma_launch_count()
    for N, T, c in ((65537, 10, cells), (10, 65537, cells), (100, 100, big)):
        with pytest.raises(H.HsmaError) as e:
            call(N, T, c)
        assert e.value.status == H.binding.HSMA_ERR_TOO_LARGE and "TOO_LARGE" in str(e.value) and "65,536" in str(e.value)
    assert H.hsma_launch_count() == launches
    src, q, tgt, out = call(65536, 65536, cells)                   # the stated maximum of N and T, 27 cells
    old = torch.empty_like(out)
    H.hsma_direct_sum(tgt, src, q, cells.shift, cells.sign, cells.w, cells.central, -1, 1, old)
    assert torch.equal(out, old)
