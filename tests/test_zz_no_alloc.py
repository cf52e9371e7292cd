"""fenc_rescale_static (-m gpu): the allocation-free rescale (include/fenc.h) against the existing path, fenc_rescale.

The two run the same three kernels over the same tables; the static call keeps its intermediates in a file-scope device
array shared by every call, so the checks are: identical limbs (the bar of every integer test here: bit-exact) on TWO
CALLS IN A ROW that reuse the array -- with different inputs, so that stale contents of the first call would show in the
second --, on both transform paths (ring degree below and from 2^12), then the same output handle overwritten again, and
the refusals (a request beyond FENC_STATIC_SCRATCH_BYTES, a wrong output handle).
Collected last on purpose (the suite runs with pytest -x); self-contained: it passes alone in a fresh process and after
the other tests."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

STATIC_SCRATCH_BYTES = 32 << 20  # FENC_STATIC_SCRATCH_BYTES in include/fenc.h


@pytest.fixture(scope="module")
def fenc():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_16359_b200 as fenc
    return fenc


@pytest.mark.parametrize("name", ["mid10", "mid12", "cfg2"])
def test_rescale_static_matches_rescale_on_two_calls_in_a_row(fenc, name):
    p = wl.PARAMS[name]
    ctx = fenc.Context(**p)
    L, N = ctx.n_q, ctx.N
    ins = [ctx.ct_import(wl.random_ct_limbs(900 + i, ctx.q, L, N), 2.0 ** 40) for i in range(3)]
    want = [ctx.ct_export(c) for c in ctx.rescale(ins)]          # the existing path, one batched call
    # output handles the caller owns: any ciphertexts at L-1 limbs (here filled with other data, to be overwritten)
    outs = [ctx.ct_import(wl.random_ct_limbs(950 + i, ctx.q, L - 1, N), 1.0) for i in range(2)]
    ctx.rescale_static_prepare(L)                                # set-up: level tables + the array's device address
    held = ctx.device_bytes()
    ctx.rescale_static(ins[0], outs[0])                          # first call
    ctx.rescale_static(ins[1], outs[1])                          # second call, same scratch array, other input
    assert ctx.device_bytes() == held                            # nothing was taken from (or returned to) the allocator
    for i in range(2):
        assert outs[i].L == L - 1
        assert np.array_equal(ctx.ct_export(outs[i]), want[i]), (name, i)
        assert abs(outs[i].scale - 2.0 ** 40 / ctx.q[L - 1]) <= 1e-9 * outs[i].scale
    ctx.rescale_static(ins[2], outs[0])                          # an output handle reused for a third input
    assert np.array_equal(ctx.ct_export(outs[0]), want[2])
    assert np.array_equal(ctx.ct_export(outs[1]), want[1])      # the other output is untouched
    # one level down: its own set-up, same array
    ctx.rescale_static_prepare(L - 1)
    low = ctx.ct_import(wl.random_ct_limbs(980, ctx.q, L - 2, N), 1.0)
    ctx.rescale_static(outs[1], low)
    assert np.array_equal(ctx.ct_export(low), ctx.ct_export(ctx.rescale([outs[1]])[0]))
    # refusals: an output at the wrong level, input and output the same ciphertext
    with pytest.raises(fenc.FencError, match="MISMATCH"):
        ctx.rescale_static(ins[0], ins[1])
    with pytest.raises(fenc.FencError, match="MISMATCH"):
        ctx.rescale_static(outs[1], outs[1])
    ctx.close()


def test_rescale_static_rejects_sizes_beyond_the_static_array(fenc):
    """A request beyond FENC_STATIC_SCRATCH_BYTES is refused, at set-up and at the call, with a message naming both sizes.
    At N = 2^16 a call needs 256 + (2 + 2 (L-1)) * 2^16 * 8 bytes: L = 31 is the largest level that fits in 32 MiB (L = 32
    needs exactly 32 MiB plus the 256-byte header); that level runs and matches the existing path."""
    N = 1 << 16
    need = lambda L: 256 + (2 + 2 * (L - 1)) * N * 8
    assert need(31) <= STATIC_SCRATCH_BYTES < need(32)
    p = dict(log2N=16, n_q=33, q_bits=50, n_p=3, p_bits=60, dnum=11, log2_scale=50)  # 11 digits of 3 limbs, P >= Q_j
    ctx = fenc.Context(**p)
    with pytest.raises(fenc.FencError, match="bytes of scratch"):
        ctx.rescale_static_prepare(33)
    big = ctx.ct_import(wl.random_ct_limbs(1, ctx.q, 33, N), 1.0)
    out = ctx.ct_import(wl.random_ct_limbs(2, ctx.q, 32, N), 1.0)
    with pytest.raises(fenc.FencError, match="bytes of scratch"):
        ctx.rescale_static(big, out)
    # the largest level that fits runs, and matches the existing path
    a = ctx.ct_import(wl.random_ct_limbs(3, ctx.q, 31, N), 1.0)
    o = ctx.ct_import(wl.random_ct_limbs(4, ctx.q, 30, N), 1.0)
    ctx.rescale_static_prepare(31)
    ctx.rescale_static(a, o)
    assert np.array_equal(ctx.ct_export(o), ctx.ct_export(ctx.rescale([a])[0]))
    ctx.close()
