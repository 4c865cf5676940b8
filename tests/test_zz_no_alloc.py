"""GPU test of voila_resample_systematic_static (include/voila.h): the resampler that allocates nothing
(scratch in a static device array of libvoila, N <= VOILA_STATIC_MAX_N = 2^20).  Its ancestors must be
those of the existing path (voila_resample_systematic, ctx workspace) bit for bit -- index work, the
tolerance of tests/test_gpu_belief.py -- on calls in a row that share the array: a large call, then a
smaller one (stale CDF / tile records behind it), then a degenerate one (status 1), then a normal one.
Collected last on purpose (the file name): the suite runs with pytest -x."""
import numpy as np
import pytest

from paper_2606_19729_b200 import synth

pytestmark = pytest.mark.gpu


def _weights(kind, N, rng):
    if kind == "skew":  # config 4: log-weights ~ N(0, 4)
        lw = 2.0 * rng.standard_normal(N)
        return np.exp(lw - lw.max()).astype(np.float32)
    if kind == "sparse":
        v = rng.uniform(0.0, 1.0, N).astype(np.float32)
        v[rng.uniform(size=N) < 0.9] = 0.0
        v[N // 2] = 1.0
        return v
    if kind == "zero":
        return np.zeros(N, np.float32)
    return rng.uniform(0.0, 1.0, N).astype(np.float32)


def test_static_resampler_matches_workspace_path(oracle):
    import torch
    import paper_2606_19729_b200 as vl
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(20)
    calls = [("skew", vl.STATIC_MAX_N, 11), ("uniform", 100_003, 12), ("zero", 5000, 13), ("sparse", 70_001, 14),
             ("uniform", 1, 15)]
    ctx = vl.Voila(synth.make_model(synth.CONFIGS[1]), device=0)
    # every buffer exists before the first call: the calls themselves must not need an allocation
    ins = [torch.from_numpy(_weights(kind, N, rng)).to(dev) for kind, N, _ in calls]
    outs = [torch.full((N,), -7, dtype=torch.int32, device=dev) for _, N, _ in calls]
    stats = [torch.full((1,), -7, dtype=torch.int32, device=dev) for _ in calls]
    refs = [ctx.voila_resample_systematic(v, seed) for v, (_, _, seed) in zip(ins, calls)]
    torch.cuda.synchronize()
    # first call: the one-time set-up (cudaGetSymbolAddress) happens here
    vl.voila_resample_systematic_static(ins[0], calls[0][2], outs[0], stats[0])
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info(dev)
    # ... the others back to back on one stream, sharing the static array
    for v, (_, _, seed), anc, st in zip(ins[1:], calls[1:], outs[1:], stats[1:]):
        vl.voila_resample_systematic_static(v, seed, anc, st)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info(dev)
    assert free1 >= free0, "the static entry point must not allocate device memory"
    for (kind, N, seed), v, anc, st, (anc_ref, st_ref) in zip(calls, ins, outs, stats, refs):
        a, r = anc.cpu().numpy(), anc_ref.cpu().numpy()
        assert int(st.item()) == int(st_ref.item()) == (1 if kind == "zero" else 0), (kind, N)
        assert np.array_equal(a, r), (kind, N)
        if kind == "zero":
            assert np.array_equal(a, np.arange(N))
        else:  # and both are the oracle's exact-integer resampler
            o, ost = oracle.resample_systematic(v.cpu().numpy(), seed)
            assert ost == 0 and np.array_equal(a, o), (kind, N)
    # the same input again after the others: the array's left-over contents do not matter
    again = torch.empty_like(outs[0])
    vl.voila_resample_systematic_static(ins[0], calls[0][2], again, None)
    torch.cuda.synchronize()
    assert torch.equal(again, outs[0])
    ctx.close()


def test_static_resampler_rejects_oversize_and_bad_arguments():
    import ctypes as C
    import torch
    import paper_2606_19729_b200 as vl
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    lib = vl.load_library()
    N = vl.STATIC_MAX_N + 1
    v = torch.ones(N, dtype=torch.float32, device="cuda:0")
    anc = torch.full((N,), -7, dtype=torch.int32, device="cuda:0")
    with pytest.raises(vl.VoilaError, match="VOILA_STATIC_MAX_N"):
        vl.voila_resample_systematic_static(v, 1, anc)
    torch.cuda.synchronize()
    assert int(anc.min().item()) == -7 and int(anc.max().item()) == -7  # nothing was launched
    rc = lib.voila_resample_systematic_static(C.c_void_p(v.data_ptr()), N, C.c_uint64(1), C.c_void_p(anc.data_ptr()),
                                              None, None)
    assert rc == 4 and b"exceeds" in lib.voila_static_last_error()  # VOILA_ERR_WORKSPACE
    rc = lib.voila_resample_systematic_static(None, 16, C.c_uint64(1), C.c_void_p(anc.data_ptr()), None, None)
    assert rc == 1  # VOILA_ERR_INVALID_ARG
    rc = lib.voila_resample_systematic_static(C.c_void_p(v.data_ptr() + 4), 16, C.c_uint64(1),
                                              C.c_void_p(anc.data_ptr()), None, None)
    assert rc == 1 and b"aligned" in lib.voila_static_last_error()
    # a good call afterwards clears the message
    vl.voila_resample_systematic_static(v[:1000], 3, anc[:1000])
    torch.cuda.synchronize()
    assert lib.voila_static_last_error() == b""
    assert int(anc[:1000].min().item()) >= 0
