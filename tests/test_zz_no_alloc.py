"""chfsi_overlap_matrix_noalloc (include/chfsi.h): S = Y^T Y with the row-split partial sums in a static device array of the
library, for callers that cannot call cudaMalloc.  `-m gpu`; collected LAST (file name) so that a failure here hides no other
test under `pytest -x`.  The reference is the existing path, chfsi_overlap_matrix (itself compared with the oracle in
test_gpu_parity.py), at the tolerance used there: 1e-12 x max |S|."""
import pytest

pytestmark = pytest.mark.gpu


def _operator(p=6, n=3):
    from paper_2203_07820_b200 import Operator
    from workloads.generate import make_workload
    wl = make_workload(None, n=n, p=p, L=2.0 * n, mesh_jitter=0.1, atoms_per_side=1, n_gaussians=0, nonlocal_=True,
                       smooth_field=0.05, seed_base=91, r_cut=2.2)
    return wl, Operator.from_workload(wl)


def test_two_calls_in_a_row_match_the_existing_path_and_allocate_nothing():
    import torch
    wl, op = _operator()
    g = torch.Generator(device="cuda")
    g.manual_seed(11)
    # call 1: N = 200 (two ragged 128-row tiles, several row splits); call 2: N = 72 on other data, so what call 1 left in
    # the static array lies exactly where call 2's partial sums go; call 3: call 1's input again
    wide = torch.randn((wl.n_dofs, 210), dtype=torch.float64, device="cuda", generator=g)
    Y1 = wide[:, 4:204]                                            # ld > N and a column offset
    Y2 = 3.0 * torch.randn((wl.n_dofs, 72), dtype=torch.float64, device="cuda", generator=g)
    ref1, ref2 = op.overlap_matrix(Y1), op.overlap_matrix(Y2)     # existing path (grows its scratch here, not below)
    S1 = torch.full((200, 200), float("nan"), dtype=torch.float64, device="cuda")
    S2 = torch.full((72, 72), float("nan"), dtype=torch.float64, device="cuda")
    S3 = torch.full((200, 200), float("nan"), dtype=torch.float64, device="cuda")
    op.overlap_matrix_noalloc(Y2, S2)                             # warm-up (first launch of the variant kernel loads its module)
    torch.cuda.synchronize()
    S2.fill_(float("nan"))
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    l0 = op.launch_count()
    op.overlap_matrix_noalloc(Y1, S1)
    op.overlap_matrix_noalloc(Y2, S2)                             # two calls in a row, same stream: ordered, no race
    op.overlap_matrix_noalloc(Y1, S3)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert op.launch_count() - l0 == 9                            # three kernels per call ran
    assert free1 >= free0, f"device memory was allocated by the allocation-free entry point: {free0 - free1} bytes"
    for S, ref in ((S1, ref1), (S2, ref2), (S3, ref1)):
        assert bool(torch.isfinite(S).all()) and torch.equal(S, S.T)
        assert float((S - ref).abs().max()) <= 1e-12 * float(ref.abs().max())
    assert torch.equal(S1, S3)                                    # deterministic, whatever the array held before
    # against the definition, too (FP64 product of torch on the device), at the same tolerance
    assert float((S2 - Y2.T @ Y2).abs().max()) <= 1e-12 * float(ref2.abs().max())
    op.close()


def test_size_limit_and_argument_errors():
    import torch
    from paper_2203_07820_b200 import ChfsiError
    wl, op = _operator(p=4, n=3)
    # at the limit: N = 512 works and agrees with the existing path
    Y = torch.randn((wl.n_dofs, 512), dtype=torch.float64, device="cuda")
    S = torch.empty((512, 512), dtype=torch.float64, device="cuda")
    op.overlap_matrix_noalloc(Y, S)
    ref = op.overlap_matrix(Y)
    assert float((S - ref).abs().max()) <= 1e-12 * float(ref.abs().max())
    # beyond it: a clear error, nothing launched
    Yb = torch.randn((wl.n_dofs, 514), dtype=torch.float64, device="cuda")
    Sb = torch.zeros((514, 514), dtype=torch.float64, device="cuda")
    l0 = op.launch_count()
    with pytest.raises(ChfsiError) as ei:
        op.overlap_matrix_noalloc(Yb, Sb)
    assert "CHFSI_NOALLOC_MAX_N = 512" in str(ei.value) and "514" in str(ei.value)
    assert op.launch_count() == l0 and float(Sb.abs().max()) == 0.0
    with pytest.raises(ChfsiError):                               # odd N: same rule as chfsi_overlap_matrix
        op.overlap_matrix_noalloc(Y[:, :33], torch.empty((33, 33), dtype=torch.float64, device="cuda"))
    op.close()


def test_the_call_can_be_captured_in_a_cuda_graph():
    """A cudaMalloc, cudaFree or synchronisation inside a stream capture is an error: capturing the call is the direct check that
    it makes none.  The graph is then replayed on new data."""
    import torch
    wl, op = _operator(p=4, n=3)
    Y = torch.randn((wl.n_dofs, 64), dtype=torch.float64, device="cuda")
    S = torch.zeros((64, 64), dtype=torch.float64, device="cuda")
    op.overlap_matrix_noalloc(Y, S)                               # warm-up outside the capture
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        op.overlap_matrix_noalloc(Y, S)                           # enqueued on the capture stream (torch's current stream)
    Y.copy_(torch.randn_like(Y))
    S.zero_()
    graph.replay()
    torch.cuda.synchronize()
    ref = op.overlap_matrix(Y)
    assert float((S - ref).abs().max()) <= 1e-12 * float(ref.abs().max())
    op.close()
