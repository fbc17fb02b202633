"""pasta_clusters_noalloc -- cluster labels for callers that cannot allocate device memory -- against pasta_clusters.

Who needs it: a process whose GPU memory is already spoken for (a framework's caching allocator or a job sized to fill
the card: cudaMalloc fails there), and an analysis thread beside a running simulation (cudaMalloc / cudaFree synchronise
the whole device and would stall the steps on the other streams).  The entry point keeps its union-find forest in a
fixed array inside the library, so it takes at most PASTA_CLUSTERS_NOALLOC_MAX_N nucleons and every call on a GPU
reuses the same memory.

The file sorts last on purpose (`pytest --collect-only`): under `pytest -x` a failure here hides no other test.  It must
pass alone in a fresh process (the first call does the per-device set-up) and after the rest of the suite.
The bar is the one tests/test_gpu_parity.py holds cluster labels to: bit-exact labels and cluster count.
"""
import ctypes as C

import pytest

import paper_1412_8502_b200 as pasta

pytestmark = pytest.mark.gpu


def _labels_both_ways(torch, N, density, r_cl, seed, label_out, n_out):
    """(labels, count) of pasta_clusters and of the no-alloc entry point on the same positions."""
    with pasta.Sim(N, 0.4, density, 1.0, seed=seed) as sim:
        ref_label, ref_n = sim.clusters(r_cl)
        x, _, _, L, _ = sim.get_state()
        torch.cuda.synchronize()
        pasta.clusters_noalloc(x, L, r_cl, label_out[:N], n_out)
        torch.cuda.synchronize()
        return ref_label.clone(), ref_n, label_out[:N].clone(), int(n_out.item())


def test_two_calls_in_a_row_match_the_allocating_path():
    import torch

    # outputs are the caller's, made once up front: a caller that cannot allocate would do the same
    label_out = torch.full((20000,), -7, dtype=torch.int32, device="cuda")
    n_out = torch.full((1,), -7, dtype=torch.int64, device="cuda")
    # first call: 20 000 nucleons; second call: fewer nucleons and another linking length, so that the forest of the
    # first call is still lying in the shared array beyond (and under) what the second one uses; third: the first again
    cases = [(20000, 0.05, 3.0, 11), (6000, 0.02, 2.4, 12), (20000, 0.05, 3.0, 11)]
    results = []
    for N, density, r_cl, seed in cases:
        ref_label, ref_n, label, n = _labels_both_ways(torch, N, density, r_cl, seed, label_out, n_out)
        assert 1 < ref_n < N  # the case has real clusters: neither one blob nor all singletons
        assert n == ref_n
        assert torch.equal(label, ref_label)
        results.append((label, n))
    assert results[0][1] == results[2][1] and torch.equal(results[0][0], results[2][0])


def test_at_the_ceiling_and_one_past_it():
    import torch

    N = pasta.CLUSTERS_NOALLOC_MAX_N
    label_out = torch.empty(N, dtype=torch.int32, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
    ref_label, ref_n, label, n = _labels_both_ways(torch, N, 0.05, 3.0, 5, label_out, n_out)
    assert n == ref_n and torch.equal(label, ref_label)

    # one nucleon more than the fixed array holds: refused by name, before anything reaches the GPU
    x = torch.zeros((N + 1, 3), dtype=torch.float64, device="cuda")
    big = torch.full((N + 1,), -3, dtype=torch.int32, device="cuda")
    with pytest.raises(pasta.PastaError) as err:
        pasta.clusters_noalloc(x, 100.0, 3.0, big)
    assert err.value.code == -1 and "PASTA_CLUSTERS_NOALLOC_MAX_N" in str(err.value) and str(N) in str(err.value)
    torch.cuda.synchronize()
    assert bool((big == -3).all())

    # the other refusals, and the empty system
    lib = pasta.load()
    ptr = C.c_void_p(x.data_ptr())
    out = C.c_void_p(big.data_ptr())
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    assert lib.pasta_clusters_noalloc(ptr, 10, 100.0, 60.0, out, None, 0, st) == -1  # r_cl > L/2
    assert lib.pasta_clusters_noalloc(None, 10, 100.0, 3.0, out, None, 0, st) == -1
    assert lib.pasta_clusters_noalloc(ptr, 10, 100.0, 3.0, out, None, 64, st) == -1
    assert lib.pasta_clusters_noalloc(None, 0, 100.0, 3.0, None, C.c_void_p(n_out.data_ptr()), 0, st) == 0
    torch.cuda.synchronize()
    assert int(n_out.item()) == 0


def test_it_allocates_nothing_on_the_device():
    """Free device memory as the driver reports it does not move across calls (after the first, which loads the
    module), and torch's allocator hands out nothing either."""
    import torch

    N = 8000
    with pasta.Sim(N, 0.4, 0.05, 1.0, seed=3) as sim:
        x, _, _, L, _ = sim.get_state()
        ref_label, ref_n = sim.clusters(3.0)
    label_out = torch.empty(N, dtype=torch.int32, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
    pasta.clusters_noalloc(x, L, 3.0, label_out, n_out)  # set-up call
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    torch_bytes0 = torch.cuda.memory_allocated()
    for _ in range(3):
        pasta.clusters_noalloc(x, L, 3.0, label_out, n_out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0 and torch.cuda.memory_allocated() == torch_bytes0
    assert int(n_out.item()) == ref_n and torch.equal(label_out, ref_label)
