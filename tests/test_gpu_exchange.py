"""SURVEY 8(e), the one exchange step of the sharded path: the covariance window of ALL ranks' chains feeds every
rank's whitening factor (best_set_adaptation_exchange).  One GPU: two 'ranks' are two contexts holding the two
halves of the chains (chain offset B), and the all-gather is stood in for by a callback that places packets
recorded from the other rank -- exact for the first window, whose samples do not depend on the exchange.  The
expected values are the oracle's covariance -> Cholesky of the pooled window and the single-process run."""
import numpy as np
import pytest

from paper_2606_04895_b200 import workloads as WL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2606_04895_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle
    oracle.lib()
    return oracle


def f32(x):
    return float(np.float32(x))


def _views(send, recv, count, world):
    from paper_2606_04895_b200.distributed import device_view
    return device_view(send, count), device_view(recv, count * world)


@pytest.mark.parametrize("prec", ["fp32", "bf16"])
def test_E_exchange_pooled_window(B, O, prec):
    import torch
    P = B.PREC_BF16 if prec == "bf16" else B.PREC_FP32
    Bk, W = 300, 40                                   # 300 chains per rank: ragged against every tile size
    w = WL.lcdm(n_chains=2 * Bk, hidden=64, n_hidden=2)
    w.L = np.diag(np.sqrt(np.diag(w.Sigma)))
    d = w.d
    npk = 1 + 2 * d + d * d

    def run(theta0, chain0, fn, world):
        ctx = B.Context(w, P)
        st = ctx.new_state(theta0)
        st.set_chain_offset(chain0)
        st.set_adaptation(W, 1e-6)
        if fn is not None:
            st.set_adaptation_exchange(fn, world)
        tr = torch.zeros(W, theta0.shape[0], d, device="cuda")
        st.step_mh(W, 33, f32(0.05), trace=tr, thin=1)
        torch.cuda.synchronize()
        L, stats = ctx.get_whitening(), ctx.adapt_stats()
        ctx.close()
        return L, stats, tr.cpu().numpy().astype(np.float64)

    # the job in one process: all 600 chains in one state
    L_all, stats, tr_all = run(w.theta0, 0, None, 1)
    assert stats == (1, 0)
    rec = {}

    def record_dummy(send, recv, count, stream):     # rank 1, first pass: record its packet, gather a dummy
        s, r = _views(send, recv, count, 2)
        assert count == npk
        rec[1] = s.clone()
        r[:count].copy_(s)
        r[count:].copy_(s)
        return 0

    def rank0(send, recv, count, stream):
        s, r = _views(send, recv, count, 2)
        rec[0] = s.clone()
        r[:count].copy_(s)
        r[count:].copy_(rec[1])
        return 0

    def rank1(send, recv, count, stream):
        s, r = _views(send, recv, count, 2)
        assert torch.equal(s, rec[1])                 # same chains, same streams: the same packet as in the first pass
        r[:count].copy_(rec[0])
        r[count:].copy_(s)
        return 0

    run(w.theta0[Bk:], Bk, record_dummy, 2)
    L0, st0, tr0 = run(w.theta0[:Bk], 0, rank0, 2)
    L1, st1, tr1 = run(w.theta0[Bk:], Bk, rank1, 2)
    assert st0 == st1 == (1, 0)
    # the shards are the job's chains (offset streams), so the pooled window is the single-process window
    assert np.array_equal(np.concatenate([tr0, tr1], axis=1), tr_all)
    # every rank ends with the same bits
    assert np.array_equal(L0, L1)
    # ... equal to the oracle's covariance -> Cholesky of the pooled samples (fp32-rounded trace: rel 1e-6, as T6)
    rc, _, Lo = O.Oracle(w).cov_chol(tr_all.reshape(-1, d), 1e-6)
    assert rc == 0
    scale = np.abs(Lo).max()
    assert np.abs(L0 - Lo).max() / scale < 1e-6
    # ... and to the single-process factor up to the summation order (fp64 sums about different reference points)
    assert np.abs(L0 - L_all).max() / scale < 1e-9
    # a rank's own window alone gives a different factor: the exchange did something
    rc, _, Lo0 = O.Oracle(w).cov_chol(tr0.reshape(-1, d), 1e-6)
    assert np.abs(L0 - Lo0).max() / scale > 1e-4
    print(f"exchange {prec}: |L - L_oracle| {np.abs(L0 - Lo).max() / scale:.2e}, |L - L_single| "
          f"{np.abs(L0 - L_all).max() / scale:.2e}")


@pytest.mark.parametrize("prec", ["fp32", "bf16"])
def test_E_exchange_world1_is_identity(B, prec):
    """world_size = 1 (the all-gather is a copy): pack -> gather -> combine -> finalize reproduces the run without an
    exchange bit for bit over several windows, through best_burn_in as well."""
    P = B.PREC_BF16 if prec == "bf16" else B.PREC_FP32
    w = WL.lcdm(n_chains=257, hidden=64, n_hidden=2)
    w.L = np.diag(np.sqrt(np.diag(w.Sigma)))
    calls = []

    def copy(send, recv, count, stream):
        s, r = _views(send, recv, count, 1)
        r.copy_(s)
        calls.append(count)
        return 0

    res = []
    for fn in (None, copy):
        ctx = B.Context(w, P)
        st = ctx.new_state(w.theta0)
        st.set_adaptation(30, 1e-6)
        if fn:
            st.set_adaptation_exchange(fn, 1)
        st.step_mala(90, 5, f32(0.05))
        eps, _, _, _ = st.burn_in("mala", 2, 60, 20, 10, 9, 0.05, 0.574)
        res.append((ctx.get_whitening(), st.get(), ctx.adapt_stats(), eps))
        ctx.close()
    (La, sa, aa, ea), (Lb, sb, ab, eb) = res
    assert aa == ab == (5, 0) and len(calls) == 5 and ea == eb
    assert np.array_equal(La, Lb)
    for k in ("theta", "logp", "grad", "n_accept"):
        assert np.array_equal(sa[k], sb[k]), k


def test_E_exchange_errors(B):
    w = WL.tiny()
    ctx = B.Context(w, B.PREC_FP32)
    st = ctx.new_state(w.theta0)
    with pytest.raises(B.BestError) as e:
        st.set_adaptation_exchange(lambda *a: 0, 0)
    assert e.value.code == B.BEST_ERR_ARG
    st.set_adaptation(10, 1e-6)
    st.set_adaptation_exchange(lambda *a: 7, 1)       # a failing callback fails the step call
    with pytest.raises(B.BestError) as e:
        st.step_mh(10, 1, 0.3)
    assert e.value.code == B.BEST_ERR_CUDA
    st.set_adaptation_exchange(None, 1)
    st.set_adaptation(10, 1e-6)
    st.step_mh(10, 1, 0.3)
    ctx.close()


@pytest.mark.parametrize("de", [False, True])
@pytest.mark.parametrize("prec", ["fp32", "bf16"])
def test_E_aies_sharded_two_ranks(B, prec, de):
    """best_set_aies_exchange: two 'ranks' (two contexts driven by two host threads, the all-gather a rendezvous
    between their callbacks) each move their slice of every half-ensemble; after 6 steps both hold the state of the
    unsharded run bit for bit (that run is itself checked against the oracle by the T2 / N3 tests)."""
    import threading
    import torch
    P = B.PREC_BF16 if prec == "bf16" else B.PREC_FP32
    w = WL.sterile(n_chains=600, hidden=64, n_hidden=2)        # halves of 300, slices of 150: ragged against every tile
    world, n_steps = 2, 6

    def advance(st):
        if de:
            st.step_aies_de(n_steps, 13, 0.1)
        else:
            st.step_aies(n_steps, 13, 2.0)

    ctx = B.Context(w, P)
    st = ctx.new_state(w.theta0)
    advance(st)
    ref = st.get(want_grad=False)
    ctx.close()
    assert 0.05 < ref["n_accept"].sum() / (600 * n_steps) < 0.95

    bar = threading.Barrier(world)
    slots, results, errors, calls = [None] * world, [None] * world, [], [0] * world

    def make_fn(rank):
        def fn(send, recv, count, stream):
            s, r = _views(send, recv, count, world)
            slots[rank] = s.clone()
            torch.cuda.synchronize()
            bar.wait(timeout=120)
            for k in range(world):
                r[k * count:(k + 1) * count].copy_(slots[k])
            torch.cuda.synchronize()
            bar.wait(timeout=120)                               # every rank has read before a slot is replaced
            calls[rank] += 1
            return 0
        return fn

    def worker(rank):
        try:
            c = B.Context(w, P)
            s = c.new_state(w.theta0)
            s.set_aies_exchange(make_fn(rank), rank, world)
            advance(s)
            results[rank] = s.get(want_grad=False)
            c.close()
        except Exception as e:                                  # noqa: BLE001
            errors.append(e)
            bar.abort()

    th = [threading.Thread(target=worker, args=(r,)) for r in range(world)]
    for t in th:
        t.start()
    for t in th:
        t.join(timeout=300)
    assert not errors, errors
    assert calls == [2 * n_steps] * world                       # one all-gather per half-step
    own = np.zeros((world, 600), bool)
    for r in range(world):
        own[r, 150 * r:150 * r + 150] = True                    # first half
        own[r, 300 + 150 * r:300 + 150 * r + 150] = True        # second half
    for r in range(world):
        assert np.array_equal(results[r]["theta"], ref["theta"]), r
        assert np.array_equal(results[r]["logp"], ref["logp"]), r
        assert np.array_equal(results[r]["n_accept"][own[r]], ref["n_accept"][own[r]])
        assert (results[r]["n_accept"][~own[r]] == 0).all()


def test_E_aies_exchange_errors(B):
    import torch
    w = WL.sterile(n_chains=100, hidden=64, n_hidden=2)
    ctx = B.Context(w, B.PREC_FP32)
    st = ctx.new_state(w.theta0)
    for rank, world in ((0, 3), (2, 2), (0, 0)):               # 50 walkers per half do not divide by 3; rank outside
        with pytest.raises(B.BestError) as e:
            st.set_aies_exchange(lambda *a: 0, rank, world)
        assert e.value.code == B.BEST_ERR_ARG
    st.set_aies_exchange(lambda *a: 0, 0, 2)
    tr = torch.zeros(1, 100, w.d, device="cuda")
    with pytest.raises(B.BestError) as e:
        st.step_aies(1, 1, 2.0, trace=tr, thin=1)
    assert e.value.code == B.BEST_ERR_ARG
    st.set_aies_exchange(None, 0, 1)
    st.step_aies(1, 1, 2.0, trace=tr, thin=1)
    ctx.close()


def test_E_exchanges_over_nccl_world1(B):
    """The callbacks of distributed.py over a real NCCL process group (one rank: the only size one GPU allows): the
    all-gather runs on the library's stream through torch.distributed on zero-copy views of the library's buffers,
    and both exchanges reproduce the runs without them bit for bit."""
    import socket
    import torch
    import torch.distributed as dist
    from paper_2606_04895_b200 import distributed as D
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1,
                            device_id=torch.device("cuda:0"))
    try:
        fn = D.allgather_exchange()
        w = WL.lcdm(n_chains=300, hidden=64, n_hidden=2)
        w.L = np.diag(np.sqrt(np.diag(w.Sigma)))
        side = torch.cuda.Stream()                                # a non-default stream: the callback must follow it
        res = []
        for use in (False, True):
            ctx = B.Context(w, B.PREC_BF16)
            st = ctx.new_state(w.theta0)
            st.set_adaptation(20, 1e-6)
            if use:
                st.set_adaptation_exchange(fn, 1)
            st.step_mala(60, 3, f32(0.05), stream=side.cuda_stream)
            st.set_adaptation(0)
            if use:
                st.set_aies_exchange(fn, 0, 1)
            st.step_aies(4, 8, 2.0, stream=side.cuda_stream)
            side.synchronize()
            res.append((ctx.get_whitening(), st.get(want_grad=False), ctx.adapt_stats()))
            ctx.close()
        (La, sa, aa), (Lb, sb, ab) = res
        assert aa == ab == (3, 0)
        assert np.array_equal(La, Lb)
        for k in ("theta", "logp", "n_accept"):
            assert np.array_equal(sa[k], sb[k]), k
    finally:
        dist.destroy_process_group()
