"""The no-allocation entry point: moebius_reshard_naive_static (csrc/moebius_static.cu).

Some callers cannot call cudaMalloc where they stand (CUDA graph capture, tight serving loops, harnesses
that forbid it).  For them the staged path of PAPER.md Table 1 exists with its staging buffer in a
file-scope static device array of MOEBIUS_STATIC_SCRATCH_BYTES (64 MiB) inside the library.  This file
checks the new entry point against the EXISTING path of the same kernels (moebius_reshard_naive with a
caller-owned buffer) byte for byte -- tolerance 0, like every parity test here: it is byte movement --
and against the oracle, on two calls in a row that share the array; that the second call leaves the
free device memory as it found it; and that a plan beyond the limit is refused before anything moves.

The file name sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide
the tests of the product path.  It passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

import workloads as wl
from harness import EP, TP, mb
from test_gpu_parity import SMALLISH, download, gpu_session, gpu_switch, naive_execute, start

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def static_execute(sess, plan):
    """The staged path with the library's static scratch: the caller passes no buffer at all."""
    need = mb.moebius_naive_scratch_bytes(sess.ctx, plan)
    assert need <= mb.moebius_static_scratch_bytes()
    st = mb.moebius_reshard_naive_static(sess.ctx, plan, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert st["scratch_bytes"] <= mb.moebius_static_scratch_bytes()
    return st


def run_two_switches(cfg, execute):
    """TP -> EP -> TP from seeded random tables; every switch is compared with the oracle inside
    gpu_switch; returns the unified buffer after each switch."""
    st, sess = gpu_session(cfg, fill="tag")
    owner, bt, _ = start(st, sess, TP, "random")
    mode, images = TP, []
    for _ in range(2):
        mode, owner, bt, _ = gpu_switch(st, sess, mode, owner, bt, execute=execute)
        images.append(download(sess).copy())
    sess.close()
    return images


@pytest.mark.parametrize("name", ["smallish", "replicated_heads"])
def test_static_scratch_entry_matches_the_existing_path_on_two_calls_in_a_row(name):
    cfg = {"smallish": SMALLISH,
           "replicated_heads": wl.get_config("tiny").with_(R=8, E=8, I=64, kv_heads=4, n_req=7, len_dist=("uniform", 1, 70), seed=13)}[name]
    assert mb.moebius_static_scratch_bytes() == 64 << 20
    got = run_two_switches(cfg, static_execute)        # two calls in a row on the shared array
    want = run_two_switches(cfg, naive_execute)        # the existing path: caller-owned scratch
    for k in range(2):
        assert got[k].shape == want[k].shape
        assert np.array_equal(got[k], want[k]), "switch %d: the static-scratch path differs from moebius_reshard_naive" % k


def test_static_scratch_call_allocates_no_device_memory():
    """Free device memory (cudaMemGetInfo) and torch's allocator are the same before and after a call.  The
    first call of a process is left out of the measurement: it may load the module that holds the array."""
    st, sess = gpu_session(SMALLISH.with_(L=1), fill="tag")
    owner, bt, _ = start(st, sess, TP, "random")
    stream = torch.cuda.current_stream().cuda_stream
    mode = TP
    for k in range(3):
        to = EP if mode == TP else TP
        plan = sess.plan(to, st.lens, owner, bt, from_mode=mode)
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        t0 = torch.cuda.memory_reserved()
        mb.moebius_reshard_naive_static(sess.ctx, plan, stream)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        if k > 0:
            assert free1 == free0, "call %d changed the free device memory by %d bytes" % (k, free0 - free1)
        assert torch.cuda.memory_reserved() == t0
        new_owner, bt = sess.block_tables(plan, len(st.lens))
        owner = new_owner if to == EP else None
        sess.free_plan(plan)
        mode = to
    sess.close()


def test_plan_beyond_the_static_limit_is_refused_untouched():
    """BASELINE.json config 2 needs more staging than the array holds: MOEBIUS_E_STAGING, nothing enqueued,
    the active mode and every device byte as before; the caller-owned path still takes the same plan."""
    cfg = wl.get_config("small").with_(L=1)      # the KV staging need does not depend on L: 64 requests, 263 MiB
    st, sess = gpu_session(cfg, fill="tag")
    owner, bt, _ = start(st, sess, TP, "random")
    before = download(sess).copy()
    plan = sess.plan(EP, st.lens, owner, bt, from_mode=TP)
    assert mb.moebius_naive_scratch_bytes(sess.ctx, plan) > mb.moebius_static_scratch_bytes()
    with pytest.raises(mb.MoebiusError) as e:
        mb.moebius_reshard_naive_static(sess.ctx, plan, torch.cuda.current_stream().cuda_stream)
    assert e.value.status == -3 and "staging buffer too small" in str(e.value)
    assert mb.moebius_active_mode(sess.ctx) == TP
    assert np.array_equal(download(sess), before)
    sess.free_plan(plan)
    gpu_switch(st, sess, TP, owner, bt, execute=naive_execute)
    sess.close()
