"""pcpd_run_series_static - the one entry point that allocates nothing (include/pcpd.h): pcpd_run_series with its
device-side record buffer in a fixed file-scope `static __device__` array of the library instead of a buffer taken from
the allocator on every call.  Checked against the existing path (pcpd_run_series on a twin handle) bit for bit - counts
are integers, the bar of every parity test here - on two calls in a row, the second shorter than the first so that the
first call's records are still in the shared buffer when it starts.

Collected last on purpose (the suite runs with -x); must pass alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pk():
    import paper_1301_6082_b200 as pk
    from paper_1301_6082_b200 import build

    build.build()
    return pk


def _torch_allocations():
    import torch

    return torch.cuda.memory_stats().get("allocation.all.allocated", 0)


def test_run_series_static_equals_run_series_on_two_calls_in_a_row(pk):
    L, R = 4096, 256
    kw = dict(L=L, n_replicas=R, d=0.3, p=0.12, seed=77, variant=pk.PCPD)
    a, b = pk.Pcpd(**kw), pk.Pcpd(**kw)       # a: existing path, b: static buffer
    a.init(pk.INIT_BERNOULLI)
    b.init(pk.INIT_BERNOULLI)
    first = [0, 1, 2, 3, 5, 8, 8, 13, 21]       # 9 records x 256 replicas x 2 observables
    second = [21, 22, 30]                       # shorter: the buffer still holds the first call's records
    for times in (first, second):
        ca, pa = a.run_series(times, pairs=True)
        n0 = _torch_allocations()
        cb, pb = b.run_series_static(times, pairs=True)
        assert _torch_allocations() == n0       # nothing went through the allocator the binding installs
        assert a.sweep == b.sweep == times[-1]
        assert np.array_equal(ca, cb) and np.array_equal(pa, pb)
    # one observable at a time (the other layout of the buffer), then the lattices agree as well
    assert np.array_equal(a.run_series([30, 31]), b.run_series_static([30, 31]))
    assert np.array_equal(a.get_lattice(), b.get_lattice())
    a.close()
    b.close()


def test_run_series_static_limits_and_errors(pk):
    R = 64 * 32
    g = pk.Pcpd(2048, R, 0.5, 0.15, 3, pk.PCPD)
    g.init(pk.INIT_FULL)
    n_max = pk.STATIC_SERIES_MAX_COUNTS // R                    # 256 records of 2048 counts fill the buffer exactly
    ref = pk.Pcpd(2048, R, 0.5, 0.15, 3, pk.PCPD)
    ref.init(pk.INIT_FULL)
    times = [k // 64 for k in range(n_max)]                     # sweeps 0 .. 3, many repeated records
    assert np.array_equal(g.run_series_static(times), ref.run_series(times))
    with pytest.raises(pk.PcpdError, match="exceed the maximum"):
        g.run_series_static([4] * (n_max + 1))                  # one record too many
    with pytest.raises(pk.PcpdError, match="exceed the maximum"):
        g.run_series_static([4] * (n_max // 2 + 1), pairs=True)
    assert g.sweep == 3                                          # a refused call does nothing
    with pytest.raises(pk.PcpdError):
        g.run_series_static([2])                                 # behind the counter
    g.close()
    ref.close()


def test_run_series_static_refuses_to_compile_and_works_after_a_warm_up(pk):
    """A handle large enough for the run-time specialised kernel compiles it (NVRTC, module load: both allocate) in its
    first sweep; the no-allocation entry point refuses to be that first sweep, and works once pcpd_run has been called."""
    c = wl.BY_NAME["cfg5"]
    g = pk.Pcpd(c.L, c.n_replicas, c.d, c.p, c.seed, c.variant)
    ref = pk.Pcpd(c.L, c.n_replicas, c.d, c.p, c.seed, c.variant)
    g.init(c.init)
    ref.init(c.init)
    with pytest.raises(pk.PcpdError, match="run one sweep"):
        g.run_series_static([1, 2])
    assert np.array_equal(g.run_series_static([0]), ref.run_series([0]))   # no sweep to run: nothing to compile
    g.run(1)
    ref.run(1)
    n0 = _torch_allocations()
    cg, pg = g.run_series_static([1, 2, 4], pairs=True)
    assert _torch_allocations() == n0
    cr, pr = ref.run_series([1, 2, 4], pairs=True)
    assert np.array_equal(cg, cr) and np.array_equal(pg, pr)
    g.close()
    ref.close()
