"""sa_linear_noalloc against sa_linear_ws (the existing split-K path), on a B200 through the C ABI.  Run with -m gpu.

sa_linear_noalloc exists for callers that cannot hand the library a workspace because they cannot get device memory
at all: an operator living inside another engine's fixed memory plan, a serving worker whose HBM is already taken by
the KV pool and the weights, a loop that must never reach cudaMalloc / cudaFree because either may stall the device.
Its split-K partials go to a 20 MiB array built into the library instead of a caller buffer, and every call on a
device shares that array.  So the questions here are the ones such a caller would ask:
  * is the result what sa_linear_ws gives (it runs the same kernels in the same order: bit for bit, and therefore within
    the layer tests' bf16 gate, |diff| <= 2^-8 |ref| + 1e-3 rms(ref), which is what is asserted first),
  * does a second call, on another shape and other data, still give that, with the first call's partials (and whatever
    earlier tests of this process left) still sitting in the array,
  * does a call really leave the amount of free device memory alone,
  * is a shape outside its range refused without anything being written.

The file name sorts after every other test file on purpose: pytest -x stops at the first failure, and a problem in this
add-on call must not hide the results of the parity tests.  It passes on its own in a fresh process (then its first
call is the one that looks the array up) and at the end of the whole suite."""
import pytest
import torch

from paper_2607_00151_b200 import binding as sa

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _rand(shape, seed, scale=1.0):
    g = torch.Generator(device=DEV)
    g.manual_seed(seed)
    return (torch.randn(shape, generator=g, device=DEV, dtype=torch.float32) * scale).to(torch.bfloat16)


def _within_gate(got, ref, what):
    """The element gate of tests/test_gpu_layer.py with the existing path's output as the reference."""
    g, r = got.double(), ref.double()
    assert torch.isfinite(g).all(), what
    rms = r.pow(2).mean().sqrt()
    bad = (g - r).abs() > 2.0 ** -8 * r.abs() + 1e-3 * rms
    assert not bad.any(), "%s: %d elements outside the gate" % (what, int(bad.sum()))


def _existing_path(x, w, r, M, N, K):
    nb = sa.sa_linear_workspace_bytes(M, N, K)
    assert nb > 0, "the case is meant to split"
    assert nb <= sa.SA_LINEAR_NOALLOC_SCRATCH_BYTES
    ws = torch.full((nb,), 0xFF, dtype=torch.uint8, device=DEV)
    y = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device=DEV)
    sa.sa_linear_ws(x, w, y, ws, r)
    torch.cuda.synchronize()
    return y


# two calls in a row that use the array differently: 16 tiles x 9 k slices of 25 k-steps with 64 live rows, then
# 3 tiles x 3 uneven slices with 130 rows in two m-tiles and a ragged last column tile; then the first shape again on new data
CASES = [
    (64, 4096, 14336, True, 21),
    (130, 520, 448, True, 22),
    (64, 4096, 14336, False, 23),
    (1, 4096, 4096, True, 24),
]


def test_noalloc_linear_matches_workspace_linear_call_after_call():
    inputs = []
    for M, N, K, res, seed in CASES:
        x = _rand((M, K), seed)
        w = _rand((N, K), seed + 100, K ** -0.5)
        r = _rand((M, N), seed + 200) if res else None
        inputs.append((x, w, r, _existing_path(x, w, r, M, N, K)))
    outs = [torch.full((M, N), float("nan"), dtype=torch.bfloat16, device=DEV) for M, N, _, _, _ in CASES]
    # the first call of the process may load device code and look the array up; after it, a call must not move the
    # device's free memory (every tensor it touches exists already, so torch's allocator is not involved either)
    sa.sa_linear_noalloc(inputs[0][0], inputs[0][1], outs[0], inputs[0][2])
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(0)[0]
    for (x, w, r, _), y in zip(inputs[1:], outs[1:]):
        sa.sa_linear_noalloc(x, w, y, r)      # back to back on one stream: no synchronisation between the calls
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(0)[0] == free_before, "a call changed the amount of free device memory"
    for (M, N, K, _, _), (_, _, _, want), y in zip(CASES, inputs, outs):
        what = "sa_linear_noalloc %dx%dx%d" % (M, N, K)
        _within_gate(y, want, what)
        assert torch.equal(y.view(torch.int16), want.view(torch.int16)), what + ": not the bits of sa_linear_ws"


def test_noalloc_linear_refuses_what_it_cannot_serve():
    sent = 0x7FC1
    # 32 x 16 tiles: the planner does not split this, no scratch is involved -> refused, y untouched
    M, N, K = 4096, 4096, 256
    assert sa.sa_linear_workspace_bytes(M, N, K) == 0
    x, w = _rand((M, K), 1), _rand((N, K), 2)
    y = torch.full((M, N), sent, dtype=torch.int16, device=DEV)
    with pytest.raises(sa.SAError) as e:
        sa.sa_linear_noalloc(x, w, y.view(torch.bfloat16))
    assert e.value.status == sa.SA_ERR_UNSUPPORTED
    # a single k-step cannot be cut either
    with pytest.raises(sa.SAError) as e:
        sa.sa_linear_noalloc(x[:4, :64].contiguous(), w[:, :64].contiguous(), y.view(torch.bfloat16)[:4])
    assert e.value.status == sa.SA_ERR_UNSUPPORTED
    # the shape rules of sa_linear hold here too
    with pytest.raises(sa.SAError) as e:
        sa.sa_linear_noalloc(_rand((4, 72), 1), _rand((4096, 72), 2), y.view(torch.bfloat16)[:4])
    assert e.value.status == sa.SA_ERR_UNSUPPORTED
    torch.cuda.synchronize()
    assert (y == sent).all()
    sa.sa_linear_noalloc(x[:0], w, y.view(torch.bfloat16)[:0])   # no rows: nothing to do
