"""lsm_spring_energy_static: the entry point for callers that cannot allocate GPU memory.

Who they are (include/lsm.h has the long form): code that holds particle and spring arrays on the device inside a process
whose GPU memory already belongs to one arena or framework pool, a monitor running beside asynchronous lsm_step work that
must not trigger the device-wide wait of cudaFree / cudaMalloc, a long sweep whose footprint is fixed at load time.  Every
other call of the library needs an lsm_sim handle, and lsm_create allocates; this one keeps its scratch (per-block partial
sums) in a fixed 512 KB array inside liblsm_b200.so, shared by all calls, limited to 2^28 springs.

What is checked: its U against the existing path -- lsm_read_energy on a handle built from the same arrays -- to the 1e-12
relative tolerance the energy comparisons of tests/test_gpu_parity.py use, on two calls in a row that leave different
amounts of stale data in the shared array (24 blocks of partials, then 2), then the first again (same bits: what the second
call left behind changes nothing); that the calls take no device memory; the counters; the size limit.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a problem here must not
hide the parity tests.  It passes alone in a fresh process (the first call then also does the per-device set-up) and
after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest

import paper_2201_04565_b200 as lsm
from paper_2201_04565_b200.binding import lsm_create_from_problem
from lsm_inputs import config2

RTOL_U = 1e-12      # tests/test_gpu_parity.py: np.allclose(Ug, Uo, rtol=1e-12)


def test_list_longer_than_the_static_scratch_is_rejected_before_any_cuda_call():
    """No GPU needed: the size check comes first, names the limit, and nothing is dereferenced or enqueued."""
    L = lsm.library()
    err = C.create_string_buffer(512)
    one = C.c_void_p(8)                        # non-NULL stand-ins; a rejected call must not touch them
    st = L.lsm_spring_energy_static(0, None, 2, 10, lsm.STATIC_MAX_SPRINGS + 1, one, one, one, None, None, 1.0, 1.0, None, one, None,
                                    err, len(err))
    assert st == -2 and b"LSM_STATIC_MAX_SPRINGS = 268435456" in err.value and b"268435457" in err.value
    assert L.lsm_spring_energy_static(0, None, 4, 10, 5, one, one, one, None, None, 1.0, 1.0, None, one, None, err, len(err)) == -1
    assert b"dim" in err.value
    assert L.lsm_spring_energy_static(0, None, 2, 10, 5, None, one, one, None, None, 1.0, 1.0, None, one, None, None, 0) == -1


def _state_on_device(torch, p, steps, **kw):
    """Runs the existing path and returns (its U, the device tensors the no-allocation call takes, live-spring count)."""
    g = lsm_create_from_problem(p, **kw)
    g.step(steps)
    x, _ = g.read_state()
    broken, _, nb = g.read_broken()
    U_ref = float(g.read_energy()[0][0])
    g.close()
    dev = torch.device("cuda", 0)
    t = dict(x=torch.from_numpy(x).to(dev), si=torch.from_numpy(p.spring_i).to(dev), sj=torch.from_numpy(p.spring_j).to(dev),
             k=torch.from_numpy(np.ascontiguousarray(p.k, dtype=np.float64)).to(dev),
             r0=torch.from_numpy(np.ascontiguousarray(p.r0, dtype=np.float64)).to(dev),
             broken=torch.from_numpy(broken.astype(np.uint8)).to(dev),
             U=torch.full((1,), float("nan"), dtype=torch.float64, device=dev), counts=torch.full((2,), -1, dtype=torch.int64, device=dev))
    return U_ref, t, p.spring_i.size - nb, nb


def _call(t):
    lsm.lsm_spring_energy_static(t["x"], t["si"], t["sj"], t["k"], t["r0"], t["U"], broken=t["broken"], counts=t["counts"])


@pytest.mark.gpu
def test_static_scratch_energy_matches_read_energy_on_two_calls_in_a_row():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: the product path has no CPU fallback")
    # A: 256^2 two-phase lattice, perturbed so that a few brittle springs are dead at step 0, 50 steps: ~195k springs,
    #    24 blocks of partials.  B: the 64^2 fracture problem of the parity tests after 9000 steps: ~12k springs, 2 blocks,
    #    a crack's worth of broken springs.
    pa = config2(n=256, seed=11, n_blobs=60)
    pa.x = pa.x + np.random.default_rng(5).uniform(-0.02, 0.02, pa.x.shape)
    pb = config2(n=64, seed=7, n_blobs=24, du_y=4.4e-4)
    Ua, ta, live_a, nb_a = _state_on_device(torch, pa, 50)
    Ub, tb, live_b, nb_b = _state_on_device(torch, pb, 9000, exact=True)
    assert nb_a > 0 and nb_b > 10 and Ua > 0 and Ub > 0, "both states must carry energy and broken springs"
    torch.cuda.synchronize()

    _call(ta)                                   # first call in this process if the file runs alone: includes the set-up
    free0 = torch.cuda.mem_get_info(0)[0]
    _call(tb)                                   # second call, straight after, on the same stream
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(0)[0] >= free0, "the call must not take device memory"
    got_a, got_b = float(ta["U"][0]), float(tb["U"][0])
    assert abs(got_a - Ua) <= RTOL_U * abs(Ua), (got_a, Ua)
    assert abs(got_b - Ub) <= RTOL_U * abs(Ub), (got_b, Ub)
    assert ta["counts"].tolist() == [live_a, 0] and tb["counts"].tolist() == [live_b, 0]

    # the array now holds B's two partials in front of A's stale ones: A again must give A's bits again
    ta["U"].fill_(float("nan"))
    _call(ta)
    torch.cuda.synchronize()
    assert float(ta["U"][0]) == got_a

    # without the flags the dead springs are counted in, so the flags are really read
    lsm.lsm_spring_energy_static(tb["x"], tb["si"], tb["sj"], tb["k"], tb["r0"], tb["U"], counts=tb["counts"])
    torch.cuda.synchronize()
    assert tb["counts"].tolist() == [live_b + nb_b, 0] and float(tb["U"][0]) > got_b

    # bad endpoint ids are skipped and counted, not dereferenced; uniform parameters; an empty list gives exactly zero
    sj_bad = tb["sj"].clone(); sj_bad[:3] = tb["x"].shape[0]; sj_bad[3] = -1; sj_bad[4] = tb["si"][4]
    lsm.lsm_spring_energy_static(tb["x"], tb["si"], sj_bad, 2.0, 1.0, tb["U"], counts=tb["counts"])
    torch.cuda.synchronize()
    assert tb["counts"].tolist() == [live_b + nb_b - 5, 5] and np.isfinite(float(tb["U"][0]))
    lsm.lsm_spring_energy_static(tb["x"], tb["si"][:0], tb["sj"][:0], 2.0, 1.0, tb["U"], counts=tb["counts"])
    torch.cuda.synchronize()
    assert float(tb["U"][0]) == 0.0 and tb["counts"].tolist() == [0, 0]
