"""fhe_polymul_static: the ring product for callers that cannot allocate device memory (scratch in a static device array
of the library, include/fhe.h).  Compared bit for bit (the path is integer: the tolerance of every parity test here is
equality) with fhe_polymul, the existing path with a caller-owned workspace, on two calls in a row with different inputs --
the second call finds the first call's residues in the shared array.  Collected last on purpose (the suite runs with
pytest -x): it must pass alone in a fresh process and after every other test."""
import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from gpu_util import limbs_np_to_tensor  # noqa: E402


def _lib():
    import paper_2607_05920_b200 as fhe
    return fhe


# small CUDA-core conversions, the tensor-core pipeline with the whole-transform kernel, and the three-pass transforms
@pytest.mark.parametrize("N,logQ,batch", [(1024, 128, 3), (1 << 12, 620, 5), (1 << 13, 218, 9)])
def test_static_scratch_polymul_equals_the_workspace_path_twice_in_a_row(N, logQ, batch):
    fhe = _lib()
    ctx = fhe.Context(N, logQ, 32)
    assert ctx.workspace_bytes(fhe.OP_POLYMUL, batch) <= ctx.fhe_static_scratch_bytes() == 32 << 20
    ctx.fhe_polymul_static_init()
    g = synth.rng(4242 + N)
    out = torch.empty((batch, ctx.L, N), dtype=torch.int32, device="cuda")
    for call in range(2):
        a = limbs_np_to_tensor(synth.uniform_limbs(g, (batch,), N, logQ))
        b = limbs_np_to_tensor(synth.uniform_limbs(g, (batch,), N, logQ))
        if call == 1:                                  # a smaller second batch: the rest of the array keeps stale residues
            a, b = a[: batch - 1].contiguous(), b[: batch - 1].contiguous()
        want = ctx.fhe_polymul(a, b)
        out.fill_(-1)                                  # before the sample: torch loads its own kernels lazily (98 MB on first use)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        got = ctx.fhe_polymul_static(a, b, out[: a.shape[0]])
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0, "the call changed the device's free memory"
        assert torch.equal(got, want), f"call {call}: static-scratch path differs from the workspace path"
        assert np.any(got.cpu().numpy() != -1)


def test_static_scratch_rejects_what_does_not_fit_and_leaves_the_output_alone():
    fhe = _lib()
    N, logQ = 1 << 13, 218
    ctx = fhe.Context(N, logQ, 32)
    per_item = ctx.workspace_bytes(fhe.OP_POLYMUL, 1)
    batch = ctx.fhe_static_scratch_bytes() // per_item + 2
    assert ctx.workspace_bytes(fhe.OP_POLYMUL, batch) > ctx.fhe_static_scratch_bytes()
    a = torch.zeros((batch, ctx.L, N), dtype=torch.int32, device="cuda")
    out = torch.full((batch, ctx.L, N), 7, dtype=torch.int32, device="cuda")
    with pytest.raises(fhe.FheError) as ei:
        ctx.fhe_polymul_static(a, a, out)
    assert "static scratch" in str(ei.value) and "fhe_polymul" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == 7).all())
    # the largest batch that fits still runs and agrees
    fit = batch - 2
    while ctx.workspace_bytes(fhe.OP_POLYMUL, fit) > ctx.fhe_static_scratch_bytes():
        fit -= 1
    g = synth.rng(99)
    x = limbs_np_to_tensor(synth.uniform_limbs(g, (fit,), N, logQ))
    y = limbs_np_to_tensor(synth.uniform_limbs(g, (fit,), N, logQ))
    assert torch.equal(ctx.fhe_polymul_static(x, y, out[:fit]), ctx.fhe_polymul(x, y))
