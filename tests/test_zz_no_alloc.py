"""pyjac_eval_jacobian_fd_static: the forward-difference Jacobian for callers that cannot allocate device memory.

Who needs it: a combustion / flow solver that reserved the whole GPU for its own arena when it started (a cudaMalloc
made later on its behalf fails), an integrator callback inside a time-step loop that must not go through cudaMalloc /
cudaFree because both synchronise the whole device and stall the solver's other streams, a plug-in whose host application
allows no driver allocation after initialisation.  Such a caller cannot hand pyjac_eval_jacobian_fd the scratch buffer it
asks for, so this entry point keeps the scratch in a 32 MiB array compiled into the library and the caller passes only
inputs and the output.

What is checked here, on two calls in a row that share that array: each call's Jacobians equal those of the existing
path (pyjac_eval_jacobian_fd with a caller-allocated buffer) within the tolerance of the other GPU tests -- in fact bit
for bit, both run the same kernels -- although the second call finds the first call's leftovers in the array; a batch
beyond the stated maximum is refused with PYJAC_ESCRATCH and leaves the output alone; the device's free memory does not
move across a call.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here must not hide another test) and
needs nothing from the tests before it: it builds its own handle and passes alone in a fresh process as well.
"""
import numpy as np
import pytest

from paper_1605_03262_b200 import synth

pytestmark = pytest.mark.gpu

JAC_TOL = 1e-10      # Frobenius-norm relative error per state, the Jacobian tolerance of tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def torch():
    import torch as t
    if not t.cuda.is_available():
        pytest.skip("no CUDA device")
    return t


@pytest.fixture(scope="module")
def PyJac():
    from paper_1605_03262_b200 import build
    build.build()
    from paper_1605_03262_b200.binding import PyJac as P
    return P


def _dev(torch, *arrays):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]


def _assert_same(got, ref, n, ld):
    got, ref = got.cpu().numpy().reshape(n, ld * ld), ref.cpu().numpy().reshape(n, ld * ld)
    assert np.all(np.isfinite(ref)) and np.abs(ref).max() > 0.0
    err = np.linalg.norm(got - ref, axis=1)
    assert np.all(err <= JAC_TOL * np.linalg.norm(ref, axis=1)), float(err.max())
    assert np.array_equal(got, ref)          # same kernels, same launch shapes: the header promises bit identity


@pytest.mark.parametrize("cfg", [1, 0])
def test_static_scratch_fd_matches_caller_scratch_fd_on_two_calls(torch, PyJac, cfg):
    m = synth.make_mechanism(cfg)
    pj = PyJac(m)
    ns, ld = m.n_species, m.n_species + 1
    cap = pj.fd_static_max_states()
    assert cap == (4 << 20) // pj.fd_workspace_doubles(1) and cap >= 1
    # first call fills the array to its limit; the second is a smaller batch of other states, so most of the
    # array still holds the first call's increments, perturbed states and source terms when it runs
    n1, n2 = min(cap, 700), max(1, min(cap, 700) // 3 - 1)
    rtol, atol = 1e-8, 1e-12
    T, P, Y = synth.config_states(cfg, n1 + n2)
    batches = [(T[:n1], P[:n1], Y[:n1]), (T[n1:], P[n1:], Y[n1:])]
    dev = [_dev(torch, *b) for b in batches]
    outs = [torch.full((len(b[0]), ld * ld), float("nan"), dtype=torch.float64, device="cuda") for b in batches]
    refs = [pj.eval_jacobian_fd(dT, dP, dY, rtol=rtol, atol=atol, chunk_states=len(dT)) for dT, dP, dY in dev]
    torch.cuda.synchronize()

    pj.eval_jacobian_fd_static(*dev[0], out=outs[0], rtol=rtol, atol=atol)       # first call: does the set-up
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    l0 = pj.kernel_launches()
    pj.eval_jacobian_fd_static(*dev[1], out=outs[1], rtol=rtol, atol=atol)       # second call, same array
    torch.cuda.synchronize()
    assert pj.kernel_launches() - l0 == 4                                       # one chunk: four kernels
    assert torch.cuda.mem_get_info()[0] == free_before                          # nothing was allocated or freed
    _assert_same(outs[0], refs[0], n1, ld)
    _assert_same(outs[1], refs[1], n2, ld)
    # and once more with the first batch: the array now holds the second call's leftovers
    again = torch.empty_like(outs[0])
    pj.eval_jacobian_fd_static(*dev[0], out=again, rtol=rtol, atol=atol)
    _assert_same(again, refs[0], n1, ld)


def test_static_scratch_fd_refuses_batches_beyond_its_array(torch, PyJac):
    from paper_1605_03262_b200.binding import PYJAC_ESCRATCH, PyJacError
    m = synth.make_mechanism(2)                      # 111 species: 166 states fit
    pj = PyJac(m)
    ld = m.n_species + 1
    cap = pj.fd_static_max_states()
    assert 1 <= cap < 1000
    T, P, Y = synth.config_states(2, cap + 1)
    dT, dP, dY = _dev(torch, T, P, Y)
    out = torch.full((cap + 1, ld * ld), -7.0, dtype=torch.float64, device="cuda")
    l0 = pj.kernel_launches()
    with pytest.raises(PyJacError) as e:
        pj.eval_jacobian_fd_static(dT, dP, dY, out=out)
    assert e.value.code == PYJAC_ESCRATCH and "scratch" in str(e.value)
    torch.cuda.synchronize()
    assert pj.kernel_launches() == l0 and bool((out == -7.0).all())             # nothing was enqueued
    with pytest.raises(ValueError):
        pj.eval_jacobian_fd_static(dT[:2], dP[:2], dY[:2], out=None)            # the binding allocates nothing either
    # exactly the limit is accepted, and n = 0 is a no-op
    ref = pj.eval_jacobian_fd(dT[:cap], dP[:cap], dY[:cap], chunk_states=cap)
    got = pj.eval_jacobian_fd_static(dT[:cap], dP[:cap], dY[:cap], out=out)
    assert np.array_equal(got.cpu().numpy()[:cap], ref.cpu().numpy())
    pj.eval_jacobian_fd_static(dT[:0], dP[:0], dY[:0], out=out)
