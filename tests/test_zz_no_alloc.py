"""gw_loglike_batch_noalloc (include/nsgw.h): the batched likelihood with its scratch in the library's fixed device array, for
callers that cannot allocate.  Checked against the existing path (gw_loglike_batch) at the tolerance of tests/test_gpu_parity.py
(1e-10 of max(1, |<d,h>| + <h,h>/2)) on calls in a row that share the array, plus the limits.  Collected last on purpose (the
suite runs with pytest -x); it depends on no other test and leaves nothing behind."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2509_04336_b200 import workloads as W

pytestmark = pytest.mark.gpu


def wf(spec, th):
    return O.OracleProblem(spec).waveform(th)


def dev(x):
    return torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64)).cuda()


@pytest.fixture(scope="module")
def nsgw():
    from paper_2509_04336_b200 import nsgw as N
    assert torch.cuda.is_available()
    return N


def _specs(name):
    if name == "taylorf2_2det":
        return W.config2(wf)
    if name == "phenomd_2det":
        return W.config3(wf)[0]
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1", "V1"], 4.0, 512.0, (20.0, 40.0))
    return W.make_data(spec, W.INJ_C3, 12.0, wf)


def _theta(h, B, seed):
    th = h.prior_transform_batch(dev(W.uniforms(B, 11, seed)))
    th[0] = dev(np.array(W.INJ_C3))
    if B > 5:
        th[5, 1] = 1.5            # unphysical mass ratio: -inf on both paths
    return th.contiguous()


def _assert_close(h, th, got):
    ref, parts = h.gw_loglike_batch(th, parts=True)
    ref, parts, got = ref.cpu().numpy(), parts.cpu().numpy(), got.cpu().numpy()
    fin = np.isfinite(ref)
    assert np.array_equal(fin, np.isfinite(got)) and np.array_equal(ref[~fin], got[~fin])
    scale = np.maximum(1.0, np.abs(parts[fin, 0::2]).sum(1) + 0.5 * parts[fin, 1::2].sum(1))
    err = np.abs(got[fin] - ref[fin]) / scale
    assert err.max() < 1e-10, err.max()


@pytest.mark.parametrize("name", ["taylorf2_2det", "phenomd_2det", "phenomd_3det"])
def test_noalloc_matches_existing_path_on_calls_in_a_row(nsgw, name):
    h = nsgw.Handle(_specs(name))
    sizes = [nsgw.NOALLOC_MAX_ROWS, 777, 1, 2500]       # the maximum, ragged groups, one row; each call overwrites the last one's scratch
    thetas = [_theta(h, B, 900 + B) for B in sizes]
    outs = [torch.full((B,), float("nan"), dtype=torch.float64, device="cuda") for B in sizes]
    h.gw_loglike_batch_noalloc(thetas[0], outs[0])      # first use on this device: symbol address, kernel loading
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for th, out in zip(thetas, outs):
        h.gw_loglike_batch_noalloc(th, out)
    again = torch.full_like(outs[0], float("nan"))
    h.gw_loglike_batch_noalloc(thetas[0], again)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0        # nothing was allocated on the device by the five calls
    for th, out in zip(thetas, outs):
        _assert_close(h, th, out)
    assert torch.equal(again, outs[0])                  # what the calls in between left in the array does not leak into a result
    # a second handle on the same device shares the array
    h2 = nsgw.Handle(_specs(name))
    out2 = torch.empty_like(outs[1])
    h2.gw_loglike_batch_noalloc(thetas[1], out2)
    assert torch.equal(out2, outs[1])
    # empty batch: nothing to do
    h.gw_loglike_batch_noalloc(torch.empty(0, 11, dtype=torch.float64, device="cuda"), torch.empty(0, dtype=torch.float64, device="cuda"))


def test_noalloc_rejects_sizes_beyond_the_maximum(nsgw):
    h = nsgw.Handle(_specs("taylorf2_2det"))
    B = nsgw.NOALLOC_MAX_ROWS + 1
    th = _theta(h, B, 7)
    out = torch.full((B,), 123.0, dtype=torch.float64, device="cuda")
    with pytest.raises(nsgw.NsgwError, match="NSGW_NOALLOC_MAX_ROWS = 4096"):
        h.gw_loglike_batch_noalloc(th, out)
    torch.cuda.synchronize()
    assert torch.all(out == 123.0)                      # rejected before any launch
    # a frequency grid longer than the array is sized for: 32 s x (1024 - 20) Hz = 32129 bins
    long_spec = W.make_data(W.gw_spec(W.LIKE_TAYLORF2, ["H1"], 32.0, 1024.0, (20.0, 40.0)), W.INJ_C3, 12.0, wf)
    assert long_spec["n_freq"] > nsgw.NOALLOC_MAX_BINS
    hl = nsgw.Handle(long_spec)
    th = _theta(hl, 8, 8)
    with pytest.raises(nsgw.NsgwError, match="NSGW_NOALLOC_MAX_BINS = 16384"):
        hl.gw_loglike_batch_noalloc(th, torch.empty(8, dtype=torch.float64, device="cuda"))
    assert hl.gw_loglike_batch(th).shape == (8,)         # the existing path takes it
    # a handle without a GW likelihood
    spec1, smp1, _ = W.config1()
    h1 = nsgw.Handle(spec1, smp1, seed=1)
    with pytest.raises(nsgw.NsgwError):
        h1.gw_loglike_batch_noalloc(torch.zeros(4, 11, dtype=torch.float64, device="cuda"), torch.empty(4, dtype=torch.float64, device="cuda"))
