"""sw_cluster_stats_static: the cluster statistics for callers that may not allocate device memory.

Some users of libsw.so cannot let it call cudaMalloc: their process gave the whole GPU to its own memory pool at
start-up, or the measurement sits in a loop that cannot afford the device-wide stall of an allocation, or the job's
memory budget is fixed once the library is loaded.  For them the entry point counts cluster sizes in a fixed array that
is part of the library image (4 MiB, at most 2^20 sites) instead of the 4*L*L-byte scratch the context calls allocate.

What is checked here: its output equals that of the existing path (sw_measure_clusters on a context, which is itself
compared with the oracle in test_physics_gpu.py) -- integers, so the tolerance is zero -- on calls made back to back,
including a small lattice right after a large one, so that whatever the previous call left in the shared array would
show.  The file sorts after every other test file on purpose: `pytest -x` stops at the first failure, and a failure in
this add-on must not hide the parity tests.  It needs nothing from the tests before it and passes on its own in a
fresh process as well.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1208_2080_b200 import binding, build
from paper_1208_2080_b200 import workloads as wl


@pytest.fixture(scope="module")
def libsw():
    build.build()
    return binding.lib()


def test_sizes_beyond_the_static_scratch_are_refused(libsw):
    """No device needed: the size check comes before any CUDA call, and the message names the limit."""
    limit = binding.static_max_sites()
    assert limit == 1 << 20
    dummy = C.c_void_p(256)                                   # never dereferenced: the call must stop at the size check
    rc = libsw.sw_cluster_stats_static(dummy, limit + 1, dummy, None)
    assert rc == binding.ERR_INVALID_ARG
    assert b"1048576" in libsw.sw_static_last_error()
    assert libsw.sw_cluster_stats_static(None, 16, dummy, None) == binding.ERR_INVALID_ARG
    assert libsw.sw_cluster_stats_static(dummy, 16, None, None) == binding.ERR_INVALID_ARG
    with pytest.raises(binding.SwError, match="SW_STATIC_MAX_SITES"):
        binding.cluster_stats_static(256, 2048 * 2048, 256)


def _static_stats(torch, labels_host):
    """The new entry point on a copy of `labels_host` in device memory the CALLER owns (torch tensors)."""
    dev_labels = torch.from_numpy(labels_host.view(np.int32)).cuda()
    dev_out = torch.full((4,), -1, dtype=torch.int64, device="cuda")      # poisoned: the call has to overwrite all four
    stream = torch.cuda.current_stream()
    binding.cluster_stats_static(dev_labels.data_ptr(), labels_host.size, dev_out.data_ptr(), stream.cuda_stream)
    stream.synchronize()
    n_clusters, largest, sum_sq, bad = (int(v) for v in dev_out.cpu().numpy().view(np.uint64))
    return {"n_clusters": n_clusters, "largest_cluster": largest, "sum_sq": sum_sq}, bad


@pytest.mark.gpu
def test_static_scratch_matches_the_allocating_path_on_calls_in_a_row():
    torch = pytest.importorskip("torch")
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    K_c = wl.CONFIGS["c1_L256_q2"]["K"]
    # L = 1024 fills the static array to its last word; 256 after it re-uses the front of an array full of old counts;
    # 201 and 200 are not multiples of the tile size (generic kernels); 201^2 = 40401 ends in a ragged 16-site group
    for L, q, K, sweeps in ((1024, 2, K_c, 3), (256, 2, K_c, 2), (512, 3, 1.0, 2), (201, 2, 0.3, 2), (200, 4, 5.0, 2)):
        sim = binding.SwendsenWang(L, q, K, seed=1208_2080 + L)
        sim.init("random")
        for _ in range(sweeps):                              # every sweep: a new labeling, the next call in the row
            sim.sweep(1)
            want = sim.measure_clusters()                    # the existing path (its scratch: cudaMalloc / workspace)
            labels = sim.get_labels()
            got, bad = _static_stats(torch, labels)
            assert bad == 0
            assert got == want, (L, q, K)
            assert got["n_clusters"] == int(np.count_nonzero(labels == np.arange(L * L, dtype=np.uint32)))
            again, bad = _static_stats(torch, labels)        # same input twice in a row: same answer, nothing accumulates
            assert bad == 0 and again == want
        sim.close()


@pytest.mark.gpu
def test_static_scratch_edge_cases():
    torch = pytest.importorskip("torch")
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    # one cluster of all sites, right after the array was filled with other counts; then all singletons
    n = binding.static_max_sites()
    got, bad = _static_stats(torch, np.zeros(n, dtype=np.uint32))
    assert bad == 0 and got == {"n_clusters": 1, "largest_cluster": n, "sum_sq": n * n}
    got, bad = _static_stats(torch, np.arange(1000, dtype=np.uint32))
    assert bad == 0 and got == {"n_clusters": 1000, "largest_cluster": 1, "sum_sq": 1000}
    # labels that cannot be canonical roots are reported in out[3] and kept out of the counts (and out of the array)
    labels = np.zeros(64, dtype=np.uint32)
    labels[10] = 7                 # 7 is not its own label
    labels[11] = 4_000_000_000     # beyond the lattice
    got, bad = _static_stats(torch, labels)
    assert bad == 2 and got == {"n_clusters": 1, "largest_cluster": 62, "sum_sq": 62 * 62}
    # an empty lattice gives zeros; host memory is refused, not dereferenced
    dev_out = torch.full((4,), -1, dtype=torch.int64, device="cuda")
    dev_labels = torch.zeros(16, dtype=torch.int32, device="cuda")
    binding.cluster_stats_static(dev_labels.data_ptr(), 0, dev_out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert dev_out.cpu().tolist() == [0, 0, 0, 0]
    host = np.zeros(16, dtype=np.uint32)
    with pytest.raises(binding.SwError, match="device memory"):
        binding.cluster_stats_static(host.ctypes.data, 16, dev_out.data_ptr())
