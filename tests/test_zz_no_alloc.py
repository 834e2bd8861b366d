"""sc_prefill_layer_static: the prefill layer for callers that may not allocate device memory.

Two kinds of caller are meant.  A serving worker in the paper's setting has donated every spare byte
of HBM to the block pool, so a later cudaMalloc has nothing to hand out and
sc_pool_create's scratch allocation fails.  And a process that is serving right now cannot afford the
call even if it would succeed, because cudaMalloc / cudaFree wait for the whole device and stall every
stream on it.  For them the library keeps the split-KV partials in a fixed array inside its own device
image (SC_STATIC_SCRATCH_BYTES, one per GPU) and needs no sc_pool_t.

What is checked: the output of the new entry point against the regular path (sc_prefill_layer, FUSED,
mma.sync engine, same partition) within the tolerance of the other GPU tests -- and bit for bit, since
the kernels and the partition are the same and only the home of the partials differs -- on two calls
made back to back, then on a smaller call that finds the larger call's partials still in the array,
and that a request beyond the array is refused before anything is launched.

This file sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides no
other test.  It does not depend on what ran before it (the array may hold zeros, in a fresh process, or
another test's leftovers; neither is read)."""
import numpy as np
import pytest
import torch

from paper_2606_16135_b200 import binding as sc
from paper_2606_16135_b200 import build as sc_build
from paper_2606_16135_b200 import inputs as I
from paper_2606_16135_b200.runtime import bits_to_torch, torch_to_bits


@pytest.fixture(scope="module", autouse=True)
def _built():
    sc_build.build()


def _assert_within_test_tolerance(got_bits, ref_bits, what):
    """The regular path's bf16 output plays the role the oracle plays elsewhere: same bounds."""
    from gpu_util import assert_close
    assert_close(got_bits, I.bf16_bits_to_f32(ref_bits).astype(np.float64), what)


def _static_layer(c, l, tiles_per_split, out, with_new=True):
    """Enqueue the no-allocation entry point for layer l of a gpu_util.Case on the current stream."""
    q, _, _, kn, vn = c.data[l]
    dq, dk, dv = (bits_to_torch(x, c.sess.device) for x in (q, kn, vn))
    sc.sc_prefill_layer_static(c.sess.cfg, c.sess.pool_mem.data_ptr(), l, dq.data_ptr(),
                               dk.data_ptr() if with_new else 0, dv.data_ptr() if with_new else 0,
                               c.table_dev.data_ptr(), len(c.table), c.T_h, c.n, tiles_per_split,
                               out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    return dq, dk, dv          # keep the inputs alive until the caller synchronises


@pytest.mark.gpu
def test_static_scratch_entry_point_matches_the_regular_path_twice_in_a_row():
    from gpu_util import Case, assert_close

    # 1 756 keys = 28 tiles of 64; 4 tiles per partition = 7 partitions
    big = Case(L=2, Hq=4, Hkv=2, D=128, T_h=1500, n=256, NB=128, seed=9100, variant="peaked",
               engine=sc.SC_ENGINE_MMA_SYNC, split_tiles=4)
    # the new tokens go into the pool through the new entry point first (the regular path then
    # rewrites the same bytes), two layers = two calls in a row with no synchronisation between them
    outs = [torch.zeros((big.n, big.Hq, big.D), dtype=torch.bfloat16, device=big.sess.device) for _ in range(2)]
    keep = [_static_layer(big, l, 4, outs[l]) for l in range(2)]
    torch.cuda.synchronize()
    for l in range(2):
        got = torch_to_bits(outs[l])
        k, v = big.sess.read_tokens(l, 0, big.table_dev, big.T_h, big.n)       # scattered bit for bit
        assert np.array_equal(torch_to_bits(k), big.data[l][3]) and np.array_equal(torch_to_bits(v), big.data[l][4])
        ref = big.run_layer(l, sc.SC_ATTN_FUSED)                              # the existing path
        _assert_within_test_tolerance(got, ref, f"static vs regular, layer {l}")
        assert np.array_equal(got, ref), f"layer {l}: same kernels, same partition, different bits"
        assert_close(got, big.oracle_layer(l), f"static vs oracle, layer {l}")
    del keep

    # a smaller call right after: 2 partitions, so partitions 2..6 of the array still hold the big
    # call's rows; new tokens already in the pool this time (k_new = v_new = NULL)
    small = Case(L=1, Hq=2, Hkv=2, D=64, T_h=70, n=40, NB=16, seed=9200, engine=sc.SC_ENGINE_MMA_SYNC,
                 split_tiles=1)
    ref = small.run_layer(0, sc.SC_ATTN_FUSED)
    out = torch.zeros((small.n, small.Hq, small.D), dtype=torch.bfloat16, device=small.sess.device)
    keep = _static_layer(small, 0, 1, out, with_new=False)
    torch.cuda.synchronize()
    got = torch_to_bits(out)
    _assert_within_test_tolerance(got, ref, "small call after a large one")
    assert np.array_equal(got, ref)
    assert_close(got, small.oracle_layer(0), "small call vs oracle")

    # the library's own choice of partition (0): another partition than the regular path's, so the
    # comparison is within tolerance only
    out2 = torch.zeros_like(outs[0])
    keep = _static_layer(big, 1, 0, out2)
    torch.cuda.synchronize()
    _assert_within_test_tolerance(torch_to_bits(out2), torch_to_bits(outs[1]), "automatic partition")
    assert_close(torch_to_bits(out2), big.oracle_layer(1), "automatic partition vs oracle")
    del keep
    small.close()
    big.close()


def test_request_beyond_the_static_scratch_is_refused_before_any_device_work():
    """8 partitions x 256 new tokens x 32 heads x (128 + 2) floats = 34.1 MB > 32 MiB.  The check is
    host arithmetic and comes before the first CUDA call, so the pointers are never touched (and this
    test needs no GPU); 7 partitions would fit."""
    cfg = sc.make_config(32, 32, 32, 128, 16, 64, 0, 256)
    fake = 1 << 20          # non-NULL, 1024-byte aligned, never dereferenced
    with pytest.raises(sc.SwiftCacheError) as e:
        sc.sc_prefill_layer_static(cfg, fake, 0, fake, fake, fake, fake, 32, 256, 256, 1, fake, 0)
    assert e.value.status == sc.SC_ERR_CAPACITY
    assert "SC_STATIC_SCRATCH_BYTES" in str(e.value) and str(sc.SC_STATIC_SCRATCH_BYTES) in str(e.value)
    need = 8 * 256 * 32 * (128 + 2) * 4
    assert need > sc.SC_STATIC_SCRATCH_BYTES >= 7 * 256 * 32 * (128 + 2) * 4
    assert str(need) in str(e.value)
    # argument errors are reported the same way as everywhere else in the ABI
    with pytest.raises(sc.SwiftCacheError) as e:
        sc.sc_prefill_layer_static(cfg, fake, 0, fake, fake, 0, fake, 32, 256, 256, 1, fake, 0)
    assert e.value.status == sc.SC_ERR_INVALID_ARG
    with pytest.raises(sc.SwiftCacheError) as e:
        sc.sc_prefill_layer_static(cfg, fake, 0, fake, fake, fake, fake, 31, 256, 256, 0, fake, 0)
    assert e.value.status == sc.SC_ERR_CAPACITY          # table too short
