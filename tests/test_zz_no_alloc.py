"""whp_argmin_static (include/whp.h): the entry point that allocates nothing — D7 with its
per-block scratch in a static __device__ array — against the existing whp_argmin, which keeps its
scratch in the context's cudaMalloc'ed buffer. Indices and values are compared for equality (the
bar of every argmin test here: an index is an integer, the value is an element of the input).

Every case makes two calls in a row: the static array is shared by all calls and keeps the last
call's contents, so the second call runs on whatever the first one left behind (including, in one
case, a ticket the test poisons on purpose by a call of a different size).

The file sorts last on purpose (`pytest --collect-only`): a failure here under `pytest -x` hides
no other test. It passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

from paper_2110_13693_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2110_13693_b200 import whp
    ctx = whp.Context.from_problem(W.make_workload("tiny").problem)  # only for whp_argmin
    yield torch, whp, ctx
    ctx.close()


def _both(torch, whp, ctx, x, stream=None):
    """(idx, val) of the existing path and of the static one on the same device tensor"""
    out = []
    for call in (ctx.argmin, whp.argmin_static):
        idx = torch.full((1,), -7, dtype=torch.int64, device="cuda")
        val = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
        call(x, idx, val, stream=stream)
        torch.cuda.synchronize()
        out.append((int(idx.item()), float(val.item())))
    return out


def _objective(torch, n, seed, ties):
    g = torch.Generator(device="cuda")
    g.manual_seed(seed)
    if ties:  # few distinct values: the minimum occurs many times, the lowest index must win
        x = torch.randint(0, 7, (n,), generator=g, device="cuda").to(torch.float64)
    else:
        x = torch.rand(n, generator=g, device="cuda", dtype=torch.float64) * 1e6
    return x


# one value; a block's chunk (4096) and its neighbours; the neighbourhood and candidate counts of
# BASELINE.json's configs (32,640 / 16,384 / 65,536); several hundred blocks with a ragged tail
SIZES = [1, 2, 255, 4095, 4096, 4097, 16384, 32640, 65536, 1_000_003]


@pytest.mark.parametrize("n", SIZES)
@pytest.mark.parametrize("ties", [False, True])
def test_static_argmin_equals_the_existing_path_twice_in_a_row(env, n, ties):
    torch, whp, ctx = env
    for rep in range(2):  # the second call finds the first call's pairs and ticket in the array
        x = _objective(torch, n, 1000 * rep + n % 977, ties)
        (i0, v0), (i1, v1) = _both(torch, whp, ctx, x)
        assert (i1, v1) == (i0, v0), f"call {rep}: static ({i1}, {v1}) != whp_argmin ({i0}, {v0})"
        xh = x.cpu().numpy()
        assert i1 == int(np.argmin(xh)) and v1 == xh[i1]  # numpy: first occurrence of the minimum


def test_minimum_in_every_block_position_and_stale_scratch(env):
    """The winner sits in the first / a middle / the last block and at a chunk's first / last
    value; between the calls the grid shrinks and grows, so stale pairs of a larger earlier call
    lie behind the ones the current call writes."""
    torch, whp, ctx = env
    n_big, n_small = 300_000, 5_000
    for n, pos in [(n_big, 0), (n_small, n_small - 1), (n_big, n_big - 1), (n_small, 4096),
                   (n_big, 4095), (n_big, 150_000), (n_small, 0), (n_big, 4096 * 73)]:
        x = torch.full((n,), 5.0, dtype=torch.float64, device="cuda")
        x[pos] = -1.0
        if pos + 1 < n:
            x[pos + 1:] = torch.where(torch.arange(n - pos - 1, device="cuda") % 3 == 0, -1.0, 5.0)
        (i0, v0), (i1, v1) = _both(torch, whp, ctx, x)
        assert (i0, v0) == (pos, -1.0) and (i1, v1) == (pos, -1.0)


def test_without_d_val_on_a_side_stream_and_back_to_back_without_sync(env):
    torch, whp, ctx = env
    s = torch.cuda.Stream()
    xs = [_objective(torch, n, 7 + k, k % 2 == 1) for k, n in enumerate([70_000, 3, 200_001, 4096])]
    idx = [torch.full((1,), -7, dtype=torch.int64, device="cuda") for _ in xs]
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        for x, i in zip(xs, idx):  # ordered on one stream: no race on the shared array
            whp.argmin_static(x, i, None, stream=s)
    s.synchronize()
    for x, i in zip(xs, idx):
        ref = torch.full((1,), -7, dtype=torch.int64, device="cuda")
        ctx.argmin(x, ref)
        torch.cuda.synchronize()
        assert int(i.item()) == int(ref.item()) == int(np.argmin(x.cpu().numpy()))


def test_allocates_nothing_and_rejects_sizes_beyond_the_maximum(env):
    torch, whp, ctx = env
    whp.argmin_static_setup()  # idempotent
    x = _objective(torch, 50_000, 3, False)
    idx = torch.zeros(1, dtype=torch.int64, device="cuda")
    whp.argmin_static(x, idx)  # set-up done: from here on no call may take device memory
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(50):
        whp.argmin_static(x, idx)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "device memory was taken during whp_argmin_static calls"
    assert int(idx.item()) == int(np.argmin(x.cpu().numpy()))

    L = whp.lib()
    assert whp.ARGMIN_STATIC_MAX_N == 16_777_216
    # one past the maximum: refused before anything is launched, with a message that names the limit
    st = L.whp_argmin_static(x.data_ptr(), whp.ARGMIN_STATIC_MAX_N + 1, idx.data_ptr(), None, None)
    assert st == whp.ERR_OUT_OF_RANGE
    msg = L.whp_static_last_error().decode()
    assert "16777216" in msg and "WHP_ARGMIN_STATIC_MAX_N" in msg
    assert L.whp_argmin_static(x.data_ptr(), 0, idx.data_ptr(), None, None) == whp.ERR_INVALID_ARG
    assert L.whp_argmin_static(None, 5, idx.data_ptr(), None, None) == whp.ERR_INVALID_ARG
    assert L.whp_argmin_static(x.data_ptr(), 5, None, None, None) == whp.ERR_INVALID_ARG
    with pytest.raises(whp.WhpError):
        whp.argmin_static(x, idx, n=0)
    # the refused calls left the array usable
    whp.argmin_static(x, idx)
    torch.cuda.synchronize()
    assert int(idx.item()) == int(np.argmin(x.cpu().numpy()))
    assert L.whp_static_last_error() == b""


def test_the_maximum_size_itself(env):
    torch, whp, ctx = env
    n = whp.ARGMIN_STATIC_MAX_N  # 128 MB of objectives, all 4096 blocks of the scratch in use
    for rep in range(2):
        x = _objective(torch, n, 99 + rep, ties=(rep == 1))
        x[n - 1] = -3.0  # the last value of the last block
        (i0, v0), (i1, v1) = _both(torch, whp, ctx, x)
        assert (i1, v1) == (i0, v0) == (n - 1, -3.0)
        x[n - 1] = 1e9
        (i0, v0), (i1, v1) = _both(torch, whp, ctx, x)
        assert (i1, v1) == (i0, v0)
        del x
