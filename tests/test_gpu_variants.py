"""GPU parity of the widened rows (SURVEY §8 f): LASER_PROB_TOKEN (probability of the emitted token,
DESIGN A2) and the vocabulary-parallel probe (laser_probe_partial / laser_probe_combine, §8 e), each
against the fp64 oracle on the same seeded inputs.  All tests need a B200 (`-m gpu`).

The vocabulary-parallel path is exercised on ONE GPU by running the G shards' partial calls one
after the other on one stream (no kernel waits for another): what is tested is every byte of the data
path - shard-local statistics, global argmax offsets, token localisation, record layout [G, N], the
merge - not cross-GPU memory visibility, which needs more than one GPU."""
import numpy as np
import pytest

from paper_2606_31580_b200 import parallel as par, workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import _parity as p
    return p


def _token_ids(w, ora, seed):
    """A mix per row: the oracle's argmax (greedy decoding), the planted token, a random token, and
    ids outside the vocabulary."""
    rng = np.random.default_rng(seed)
    N = w.N_alloc
    tok = rng.integers(0, w.V, size=N).astype(np.int64)
    kind = rng.integers(0, 4, size=N)
    am = np.where(ora.argmax >= 0, ora.argmax, 0)
    tok = np.where(kind == 0, am, tok)
    if w.planted is not None:
        tok = np.where((kind == 1) & (w.planted >= 0), w.planted, tok)
    oov = rng.random(N) < 0.05
    tok = np.where(oov, rng.choice([-1, -7, w.V, w.V + 5, 2**31 - 1], size=N), tok)
    return tok.astype(np.int32)


def _oracle_token_mode(w, ora, tok, agg):
    """Oracle result for LASER_PROB_TOKEN: token probabilities -> aggregate -> exit (tau unchanged)."""
    import oracle
    nv = w.N_valid
    pt = np.full(w.N_alloc, np.nan)
    if nv:
        pt[:nv] = oracle.token_prob(w.hidden_f32()[:nv], w.W_f32(), tok[:nv])
    conf = oracle.aggregate(np.nan_to_num(pt, nan=0.0), w.req_offsets, mode=agg)
    ex, margin = oracle.exit_mask(conf, ora.tau)
    return pt, conf, ex, margin


def _compare_token_mode(P, w, g, ora, pt, conf, ex, margin, label):
    nv = w.N_valid
    # argmax is still the row argmax
    mism = g.argmax[:nv] != ora.argmax[:nv]
    assert not (mism & ~(ora.gap2[:nv] < P.GAP_EXEMPT)).any(), f"{label}: argmax"
    assert np.all(g.argmax[nv:] == -1)
    dp = np.abs(g.pmax[:nv].astype(np.float64) - pt[:nv])
    assert np.all(dp <= P.PMAX_TOL), f"{label}: token prob error {dp.max():.3e} at row {dp.argmax()}"
    dc = np.abs(g.conf.astype(np.float64) - conf)
    assert np.all(dc <= P.CONF_TOL), f"{label}: conf error {dc.max():.3e}"
    bad = (g.exit != ex) & ~(margin <= P.MARGIN_EXEMPT)
    assert not bad.any(), f"{label}: exit mismatch on {np.nonzero(bad)[0][:8]}"
    return dict(max_ptok_err=float(dp.max()) if dp.size else 0.0, max_conf_err=float(dc.max()) if dc.size else 0.0,
                exits=int(ex.sum()), requests_exempt=int((margin <= P.MARGIN_EXEMPT).sum()))


@pytest.mark.parametrize("agg", [0, 1])
@pytest.mark.parametrize("V,d,R,L,n_alloc,var_len,mode", [
    (33000, 512, 12, 8, None, None, 0),       # one token tile, several vocabulary tiles, ragged V
    (9000, 256, 40, None, 400, (1, 16), 3),   # several token chunks (flex kernel), padding rows
    (9000, 256, 40, None, 400, (1, 16), 4),   # the same through the mixed schedule (pair + single-CTA kernels)
    (9000, 256, 40, None, 400, (1, 16), 2),   # ... and the pair kernel alone
    (1000, 64, 8, 4, None, None, 0),          # C1 shape
])
def test_token_prob_mode(P, V, d, R, L, n_alloc, var_len, mode, agg):
    """LASER_PROB_TOKEN: conf aggregates softmax(logits)[token_ids[n]] instead of the row maximum."""
    import torch
    from paper_2606_31580_b200 import binding as B
    w = wl.scaled(f"tok-V{V}", V, d, 0.05, R, L, seed=77, N_alloc=n_alloc, var_len=var_len)
    ora, rows, reqs = P.run_oracle(w)
    tok = _token_ids(w, ora, seed=5)
    pt, conf, ex, margin = _oracle_token_mode(w, ora, tok, agg)
    dev = P.to_device(w)
    probe = B.Probe(w.N_alloc, w.d, w.V, w.R, mode=mode)
    assert probe.plan["flex"] == (1 if mode == 3 else 0)
    probe.conf.fill_(-7.0); probe.argmax.fill_(-7); probe.exit.fill_(7); probe.pmax.fill_(-7.0)
    out = probe(dev["hidden"], dev["W"], dev["off"], dev["load"], B.TauParams(**w.tau_params), agg=agg,
                token_ids=torch.from_numpy(tok).cuda())
    torch.cuda.synchronize()
    g = P.GpuRun(out.conf.cpu().numpy(), out.argmax.cpu().numpy(), out.exit.cpu().numpy(),
                 out.tau.cpu().numpy(), out.pmax.cpu().numpy(), probe.plan)
    st = _compare_token_mode(P, w, g, ora, pt, conf, ex, margin, w.name)
    print(w.name, agg, st)
    # greedy decoding: token = argmax => identical to the default mode
    out2 = probe(dev["hidden"], dev["W"], dev["off"], dev["load"], B.TauParams(**w.tau_params), agg=agg,
                 token_ids=out.argmax.clone())
    torch.cuda.synchronize()
    pm_tok = out2.pmax.cpu().numpy().copy()
    out3 = probe(dev["hidden"], dev["W"], dev["off"], dev["load"], B.TauParams(**w.tau_params), agg=agg)
    torch.cuda.synchronize()
    nv = w.N_valid
    np.testing.assert_allclose(pm_tok[:nv], out3.pmax.cpu().numpy()[:nv], rtol=2e-6, atol=0)


def test_token_prob_c2_shape(P, c2_W_bits):
    """Full C2 shape, the launch configuration bench.py times: token mode on planted / random tokens."""
    import torch
    from paper_2606_31580_b200 import binding as B
    w = wl.config_c2(c2_W_bits)
    ora, rows, reqs = P.run_oracle(w)
    tok = _token_ids(w, ora, seed=6)
    pt, conf, ex, margin = _oracle_token_mode(w, ora, tok, 0)
    dev = P.to_device(w)
    probe = B.Probe(w.N_alloc, w.d, w.V, w.R)
    out = probe(dev["hidden"], dev["W"], dev["off"], dev["load"], B.TauParams(**w.tau_params),
                token_ids=torch.from_numpy(tok).cuda())
    torch.cuda.synchronize()
    g = P.GpuRun(out.conf.cpu().numpy(), out.argmax.cpu().numpy(), out.exit.cpu().numpy(),
                 out.tau.cpu().numpy(), out.pmax.cpu().numpy(), probe.plan)
    print("tok-c2", _compare_token_mode(P, w, g, ora, pt, conf, ex, margin, "tok-c2"))


def test_token_mode_needs_token_ids(P):
    import ctypes as C
    from paper_2606_31580_b200 import binding as B
    w = wl.config_c1()
    dev = P.to_device(w)
    probe = B.Probe(w.N_alloc, w.d, w.V, w.R)
    opt = B.Options(0, B.PROB_TOKEN, None)
    tp = B.TauParams(**w.tau_params)
    rc = B.lib().laser_probe_confidence_opt(
        dev["hidden"].data_ptr(), dev["W"].data_ptr(), dev["off"].data_ptr(), dev["load"].data_ptr(),
        C.byref(tp), probe.conf.data_ptr(), probe.argmax.data_ptr(), probe.exit.data_ptr(),
        C.byref(probe.dims), probe.workspace.data_ptr(), probe.workspace.numel(), None, None, None, C.byref(opt))
    assert rc == -1
    opt = B.Options(0, 5, None)
    rc = B.lib().laser_probe_confidence_opt(
        dev["hidden"].data_ptr(), dev["W"].data_ptr(), dev["off"].data_ptr(), dev["load"].data_ptr(),
        C.byref(tp), probe.conf.data_ptr(), probe.argmax.data_ptr(), probe.exit.data_ptr(),
        C.byref(probe.dims), probe.workspace.data_ptr(), probe.workspace.numel(), None, None, None, C.byref(opt))
    assert rc == -8


# ------------------------------------------------------------------------------- vocabulary-parallel
def _run_vocab_parallel(P, w, G, tok=None, agg=0, peer=False, tail=0, mode=0):
    """G virtual ranks on one GPU, one after the other on one stream."""
    import torch
    from paper_2606_31580_b200 import binding as B
    dev = P.to_device(w)
    tok_d = torch.from_numpy(tok).cuda() if tok is not None else None
    tp = B.TauParams(**w.tau_params)
    N = w.N_alloc
    stats_all = torch.full((G, N, 4), 123.0, dtype=torch.float32, device="cuda")   # poisoned
    flags = torch.zeros(G, dtype=torch.int32, device="cuda")
    shards = []
    for g in range(G):
        v0, v1 = par.shard_vocab(w.V, G, g)
        sh = B.VocabShardProbe(N, w.d, v1 - v0, w.R, v0, G, tail=tail, mode=mode)
        Wg = dev["W"][v0:v1].contiguous()
        if peer:
            pe = B.Peers()
            pe.rank, pe.world, pe.epoch = g, G, 3
            for k in range(G):           # one GPU: every "peer" buffer is the same buffer
                pe.peer_stats[k] = stats_all.data_ptr()
                pe.peer_flags[k] = flags.data_ptr()
            sh.partial(dev["hidden"], Wg, dev["off"], token_ids=tok_d, peers=pe)
        else:
            sh.partial(dev["hidden"], Wg, dev["off"], token_ids=tok_d, out=stats_all[g])
        shards.append((sh, Wg))
    launches = None
    if tail:    # one kernel per partial with the fused tail; 2 (+1 signal with peers) with a separate reduce
        launches = B.kernel_launch_count()
    sh = shards[0][0]
    sh.conf.fill_(-7.0); sh.argmax.fill_(-7); sh.exit.fill_(7); sh.pmax.fill_(-7.0)
    out = sh.combine(dev["off"], dev["load"], tp, stats_all=stats_all, agg=agg, token_prob=tok is not None,
                     wait_flags=flags if peer else None, epoch=3 if peer else 0)
    torch.cuda.synchronize()
    if peer:
        assert np.all(flags.cpu().numpy() == 3)
    return P.GpuRun(out.conf.cpu().numpy(), out.argmax.cpu().numpy(), out.exit.cpu().numpy(),
                    out.tau.cpu().numpy(), out.pmax.cpu().numpy(), sh.plan), stats_all.cpu().numpy()


@pytest.mark.parametrize("tail", [0, 2])       # reduce + push + signal in the fused kernel's tail (one kernel) / as kernels
@pytest.mark.parametrize("peer", [False, True])
@pytest.mark.parametrize("G", [1, 2, 3, 8])
@pytest.mark.parametrize("V,d,R,L,n_alloc,var_len,mode", [
    (33000, 512, 12, 8, None, None, 0),
    (9001, 256, 40, None, 400, (1, 16), 3),  # V not divisible by G, several token chunks, padding rows: the flex kernel
    (9001, 256, 40, None, 400, (1, 16), 4),  # the same through the mixed schedule (two fused kernels per partial)
])
def test_vocab_parallel_matches_oracle(P, G, peer, tail, V, d, R, L, n_alloc, var_len, mode):
    from paper_2606_31580_b200 import binding as B
    w = wl.scaled(f"vp-V{V}-G{G}", V, d, 0.05, R, L, seed=88, N_alloc=n_alloc, var_len=var_len)
    n0 = B.kernel_launch_count()
    g, stats = _run_vocab_parallel(P, w, G, peer=peer, tail=tail, mode=mode)
    pl = B.plan_query(w.N_alloc, d, par.shard_vocab(V, G, 0)[1], R, mode=mode)
    mixed = pl["mixed"]
    assert mixed == (1 if mode == 4 else 0) and pl["flex"] == (1 if mode == 3 else 0)
    fused = 2 if mixed else 1                                           # fused kernels of one partial
    per_partial = fused if tail == 0 else fused + (2 if peer else 1)    # the tail also runs in the mixed schedule's kernels
    assert B.kernel_launch_count() - n0 == G * per_partial + 1          # + the combine kernel
    ora, rows, reqs = P.run_oracle(w)
    st = P.compare(w, g, ora, rows, reqs, w.name)
    print(w.name, "peer" if peer else "collective", {k: v for k, v in st.items() if k != "plan"})
    # the shard records themselves: global argmax inside the shard's range, neutral padding rows
    nv = w.N_valid
    for k in range(G):
        v0, v1 = par.shard_vocab(V, G, k)
        a = stats[k, :, 2].view(np.int32)
        assert np.all((a[:nv] >= v0) & (a[:nv] < v1))
        assert np.all(a[nv:] == 2**31 - 1) and np.all(np.isneginf(stats[k, nv:, 0])) and np.all(stats[k, nv:, 1] == 0)


def test_vocab_parallel_token_mode_and_ties(P):
    """Token mode across shards (the token's logit lives in exactly one shard) and a tie between two
    shards (duplicate winning rows of W in different shards: the lower global index wins)."""
    G = 4
    w = wl.scaled("vp-tok", 20000, 256, 0.05, 10, 8, seed=89)
    ora, rows, reqs = P.run_oracle(w)
    tok = _token_ids(w, ora, seed=9)
    g, _ = _run_vocab_parallel(P, w, G, tok=tok, agg=1)
    pt, conf, ex, margin = _oracle_token_mode(w, ora, tok, 1)
    print("vp-tok", _compare_token_mode(P, w, g, ora, pt, conf, ex, margin, "vp-tok"))
    # tie across shards: copy the winning row of request 0's first token into a later shard
    Wb = w.W_bits.copy()
    v1 = int(ora.argmax[0])
    v2 = (v1 + 3 * (w.V // G)) % w.V
    lo, hi = min(v1, v2), max(v1, v2)
    Wb[hi] = Wb[lo] = w.W_bits[v1]
    w2 = wl.Workload("vp-tie", Wb, w.hidden_bits, w.req_offsets, w.load, w.tau_params)
    g2, _ = _run_vocab_parallel(P, w2, G)
    ora2, rows2, reqs2 = P.run_oracle(w2)
    assert ora2.argmax[0] == lo and ora2.gap2[0] == 0.0
    assert g2.argmax[0] == lo            # bit-identical logits in both shards: exact tie on the GPU too
    P.compare(w2, g2, ora2, rows2, reqs2, "vp-tie")


def test_vocab_parallel_c2_shape(P, c2_W_bits):
    """C2 at G = 8: each virtual rank streams 1/8 of the LM head (the tensor-parallel layout)."""
    w = wl.config_c2(c2_W_bits)
    g, _ = _run_vocab_parallel(P, w, 8, peer=True)
    ora, rows, reqs = P.run_oracle(w)
    st = P.compare(w, g, ora, rows, reqs, "vp-c2-G8")
    print("vp-c2-G8", {k: v for k, v in st.items() if k != "plan"})


@pytest.mark.parametrize("exchange", ["collective", "peer"])
def test_vocab_parallel_process_group_world1(P, exchange):
    """parallel.VocabParallelProbe end to end inside a real torch.distributed NCCL group (world size 1,
    the only size one GPU allows): all-gather exchange, and the peer-push exchange over
    torch symmetric memory (peer-mapped buffers, epoch flags, two buffer sets alternating)."""
    import socket
    import os
    import torch
    import torch.distributed as dist
    from paper_2606_31580_b200 import binding as B
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dev0 = torch.device("cuda", torch.cuda.current_device())
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev0)
    try:
        w = wl.scaled("vp-pg", 9001, 256, 0.05, 40, None, seed=88, N_alloc=400, var_len=(1, 16))
        dev = P.to_device(w)
        ora, rows, reqs = P.run_oracle(w)
        vp = par.VocabParallelProbe(dist, w.N_alloc, w.d, w.V, w.R, dev0, exchange=exchange, debug_outputs=True)
        Wg = dev["W"][vp.v0:vp.v1].contiguous()
        side = torch.cuda.Stream()
        for it in range(5):      # several epochs: both buffer sets are reused; odd ones on a side stream
            vp.shard.conf.fill_(-7.0); vp.shard.argmax.fill_(-7); vp.shard.exit.fill_(7)
            torch.cuda.synchronize()
            out = vp(dev["hidden"], Wg, dev["off"], dev["load"], B.TauParams(**w.tau_params),
                     stream=side if it % 2 else None)
            torch.cuda.synchronize()
            g = P.GpuRun(out.conf.cpu().numpy(), out.argmax.cpu().numpy(), out.exit.cpu().numpy(),
                         out.tau.cpu().numpy(), out.pmax.cpu().numpy(), vp.shard.plan)
            P.compare(w, g, ora, rows, reqs, f"vp-pg-{exchange}-{it}")
        if exchange == "peer":
            assert vp.peers.epoch == 5
    finally:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------- K-block-major W
@pytest.mark.parametrize("V,d", [(1000, 64), (33000, 512), (70001, 72), (17, 8), (5000, 200)])
def test_pack_w_layout(V, d):
    """laser_probe_pack_w against the layout's definition, bit for bit: out[kb][v][c] = W[v][64 kb + c],
    zero where 64 kb + c >= d."""
    import torch
    from paper_2606_31580_b200 import binding as B
    g = torch.Generator(device="cuda").manual_seed(V + d)
    W = torch.randn((V, d), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16)
    packed = B.pack_w(W)
    kb = -(-d // 64)
    assert packed.numel() == kb * V * 64
    ref = torch.zeros((V, kb * 64), dtype=torch.bfloat16, device="cuda")
    ref[:, :d] = W
    ref = ref.view(V, kb, 64).permute(1, 0, 2).contiguous().view(-1)
    torch.cuda.synchronize()
    assert torch.equal(packed.view(torch.int16), ref.view(torch.int16))


@pytest.mark.parametrize("mode", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("V,d,R,L,n_alloc,var_len", [
    (33000, 512, 40, None, 400, (1, 16)),   # several token tiles / chunks, padding rows
    (70001, 72, 12, 8, None, None),         # d not a multiple of 64: zero columns in the packed copy, odd V
    (5000, 200, 3, 60, None, None),         # N = 180, V not a multiple of the tile heights
])
def test_kblocked_w_matches_oracle(P, mode, V, d, R, L, n_alloc, var_len):
    """Every kernel variant with W given K-block-major (laser_probe_options.w_layout): boxes that run past
    row V of a k-block slab read the next slab's rows, which the epilogue masks like TMA's zero fill."""
    from paper_2606_31580_b200 import binding as B
    w = wl.scaled(f"kblocked-m{mode}-V{V}-d{d}", V, d, 0.05, R, L, seed=V + d + 3, N_alloc=n_alloc, var_len=var_len)
    P.CFG.update(mode=mode, w_layout=B.W_KBLOCKED)
    try:
        st = P.check(w)
    finally:
        P.CFG.update(mode=0, w_layout=0)
    print(w.name, {k: v for k, v in st.items() if k != "plan"})


def test_kblocked_w_ties_at_the_slab_boundary(P):
    """Duplicate winning rows at the very end of the vocabulary (the last box runs into the next k-block
    slab) and across a tile boundary, K-block-major W: the lowest index wins, rows past V never do."""
    from paper_2606_31580_b200 import binding as B
    V, d, N = 9001, 128, 16
    rng = np.random.default_rng(21)
    Wf = (rng.standard_normal((V, d)) * 0.05).astype(np.float32)
    h = rng.standard_normal((N, d)).astype(np.float32)
    big = (h[0] * 0.5).astype(np.float32)
    P.CFG.update(w_layout=B.W_KBLOCKED)
    try:
        for v1, v2 in [(V - 2, V - 1), (207, 208), (3, V - 1)]:
            W2 = Wf.copy(); W2[v1] = big; W2[v2] = big
            w = wl.Workload("ties-kblocked", wl.bf16_bits(W2), wl.bf16_bits(h), wl.fixed_offsets(2, 8),
                            np.array([0.3, 0.7], np.float32))
            g = P.run_gpu(w)
            assert g.argmax[0] == v1, (v1, v2, g.argmax[0])
            ora, rows, reqs = P.run_oracle(w)
            assert ora.argmax[0] == v1 and ora.gap2[0] == 0.0
            P.compare(w, g, ora, rows, reqs, "ties-kblocked")
    finally:
        P.CFG.update(w_layout=0)


# ------------------------------------------------------------------------------- seeded shape fuzz
def _fuzz_case(i):
    rng = np.random.default_rng(4242 + i)
    V = int(rng.choice([rng.integers(1, 300), rng.integers(300, 5000), rng.integers(5000, 40000)]))
    d = 8 * int(rng.integers(1, 65))
    R = int(rng.integers(1, 41))
    lo = int(rng.integers(0, 3))
    hi = lo + int(rng.integers(0, 20))
    pad = int(rng.choice([0, 0, 1, 7, 130, 300]))
    mode = int(rng.integers(0, 3))
    agg = int(rng.integers(0, 3))
    if i % 3 == 2:
        mode = 3 + (i % 2)          # flex / mixed
    return V, d, R, (lo, hi), pad, mode, agg


@pytest.mark.parametrize("i", range(32))
def test_fuzz_shapes_modes_aggregates(P, i):
    """32 seeded random shapes (V 1..40000, d 8..512, ragged requests incl. empty ones, padding rows)
    x kernel variant (auto / single / pair) x aggregate, each against the oracle."""
    from paper_2606_31580_b200 import binding as B
    V, d, R, var_len, pad, mode, agg = _fuzz_case(i)
    w0 = wl.scaled(f"fuzz{i}", V, d, 0.05, R, None, seed=9000 + i, var_len=var_len)
    w = wl.scaled(f"fuzz{i}-V{V}-d{d}-R{R}-m{mode}-a{agg}", V, d, 0.05, R, None, seed=9000 + i, var_len=var_len,
                  N_alloc=w0.N_valid + pad)
    if w.N_alloc == 0:
        pytest.skip("empty batch (covered by test_empty_batches_and_requests)")
    tail, use_handle = [(0, True), (2, True), (2, False), (0, False)][i % 4]
    P.CFG.update(mode=mode, tail=tail, use_handle=use_handle)
    try:
        st = P.check(w, agg=agg)
    finally:
        P.CFG.update(mode=0, tail=0, use_handle=True)
    print(w.name, {k: v for k, v in st.items() if k != "plan"},
          "flex" if st["plan"]["flex"] else ("mixed" if st["plan"]["mixed"] else ("pair" if st["plan"]["cta_pair"] else "single")))


# ------------------------------------------------------------------------------- boundary: handles, options, debug
def test_handle_reuse_across_buffers(P):
    """One handle called with more hidden / W buffers than its descriptor cache holds (2 / 4 entries,
    round robin): every call must use the descriptors of ITS buffers."""
    import torch
    from paper_2606_31580_b200 import binding as B
    ws = [wl.scaled(f"reuse{i}", 9000, 128, 0.05, 6, 8, seed=700 + i) for i in range(6)]
    devs = [P.to_device(w) for w in ws]
    oras = [P.run_oracle(w) for w in ws]
    pr = B.Probe(ws[0].N_alloc, ws[0].d, ws[0].V, ws[0].R)
    tp = B.TauParams(**ws[0].tau_params)
    for k in [0, 1, 2, 3, 4, 5, 0, 5, 1, 4, 2, 3, 3, 0]:
        dv = devs[k]
        out = pr(dv["hidden"], dv["W"], dv["off"], dv["load"], tp)
        torch.cuda.synchronize()
        g = P.GpuRun(out.conf.cpu().numpy(), out.argmax.cpu().numpy(), out.exit.cpu().numpy(),
                     out.tau.cpu().numpy(), out.pmax.cpu().numpy(), pr.plan)
        ora, rows, reqs = oras[k]
        P.compare(ws[k], g, ora, rows, reqs, f"reuse buffer set {k}")
    assert len(pr._handles) == 1


def test_two_threads_with_different_options(P):
    """Options are per call: two host threads probe concurrently on their own streams, one forcing
    the single-CTA kernel with the fused tail, the other the pair kernel with a separate finalize."""
    import threading
    import torch
    from paper_2606_31580_b200 import binding as B
    w = wl.scaled("threads", 33000, 256, 0.05, 30, 8, seed=55)
    dev = P.to_device(w)
    ora, rows, reqs = P.run_oracle(w)
    tp = B.TauParams(**w.tau_params)
    results, errors = {}, []

    def worker(name, **kw):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            pr = B.Probe(w.N_alloc, w.d, w.V, w.R, **kw)
            for _ in range(40):
                out = pr(dev["hidden"], dev["W"], dev["off"], dev["load"], tp, stream=st)
            st.synchronize()
            results[name] = (P.GpuRun(out.conf.cpu().numpy(), out.argmax.cpu().numpy(), out.exit.cpu().numpy(),
                                      out.tau.cpu().numpy(), out.pmax.cpu().numpy(), pr.plan), pr.plan)
        except Exception as e:          # noqa: BLE001
            errors.append((name, repr(e)))

    ts = [threading.Thread(target=worker, args=("single-tail",), kwargs=dict(mode=B.MODE_SINGLE, tail=B.TAIL_FUSED)),
          threading.Thread(target=worker, args=("pair-separate",), kwargs=dict(mode=B.MODE_PAIR, tail=B.TAIL_SEPARATE)),
          threading.Thread(target=worker, args=("implicit",), kwargs=dict(use_handle=False, overlap=True))]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errors, errors
    assert results["single-tail"][1]["cta_pair"] == 0 and results["pair-separate"][1]["cta_pair"] == 1
    for name, (g, _) in results.items():
        P.compare(w, g, ora, rows, reqs, name)


@pytest.mark.parametrize("n_streams", [2, 3])
@pytest.mark.parametrize("N,R,mode", [(4096, 512, 0),      # R far above the grid: without the cap every CTA was a finalizer
                                      (1152, 144, 4)])     # nine 128-row tiles: both kernels of the mixed schedule busy, fixed finalizers
def test_concurrent_fused_tails_on_several_streams(P, n_streams, N, R, mode):
    """Fused-tail calls with more requests than the grid has CTAs, issued on two / three streams at once
    (one of them high priority), 200 calls per stream.  The CTAs of the grids interleave on the SMs; the
    finalizers of each call (at most 32) spin for CTAs that may not be resident yet, which is safe only
    while enough SMs stay free for those - the reason for the cap (include/laser_probe.h, thread-safety
    paragraph).  Every stream's result must equal the one the same handle gives alone, no trap."""
    import torch
    from paper_2606_31580_b200 import binding as B
    w = wl.scaled(f"conc-N{N}", 5000, 64, 0.05, R, N // R, seed=71 + N)
    dev = P.to_device(w)
    tp = B.TauParams(**w.tau_params)
    ora, rows, reqs = P.run_oracle(w)
    streams = [torch.cuda.Stream(priority=-1 if i == 0 else 0) for i in range(n_streams)]    # -1: high priority
    probes = [B.Probe(w.N_alloc, w.d, w.V, w.R, tail=B.TAIL_FUSED, mode=mode) for _ in range(n_streams)]
    assert probes[0].plan["kernel_launches"] == (2 if probes[0].plan["mixed"] else 1)      # fused tail: no finalize kernel
    # serial reference through the first probe
    ref = probes[0](dev["hidden"], dev["W"], dev["off"], dev["load"], tp)
    torch.cuda.synchronize()
    want = [t.cpu().numpy().copy() for t in (ref.conf, ref.argmax, ref.exit, ref.pmax)]
    g = P.GpuRun(want[0], want[1], want[2], ref.tau.cpu().numpy(), want[3], probes[0].plan)
    P.compare(w, g, ora, rows, reqs, w.name)
    for p in probes:
        p.conf.fill_(-7.0); p.argmax.fill_(-7); p.exit.fill_(7); p.pmax.fill_(-7.0)
    torch.cuda.synchronize()
    for _ in range(200):
        for p, st in zip(probes, streams):
            p(dev["hidden"], dev["W"], dev["off"], dev["load"], tp, stream=st)
    torch.cuda.synchronize()          # a trap (the 4 s watchdog of a starved finalizer) would surface here
    for i, p in enumerate(probes):
        got = [t.cpu().numpy() for t in (p.conf, p.argmax, p.exit, p.pmax)]
        for a, b, name in zip(got, want, ("conf", "argmax", "exit", "pmax")):
            assert np.array_equal(a, b, equal_nan=(name in ("conf", "pmax"))), f"stream {i}: {name}"
        p.close()


def test_debug_build_checks_req_offsets():
    """LASER_DEBUG=1: a non-monotone req_offsets makes the validation kernel trap (the call surfaces
    as a CUDA error); a valid one passes.  Run in child processes: a trap kills the CUDA context."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    prog = r"""
import sys, numpy as np, torch
sys.path.insert(0, %r)
from paper_2606_31580_b200 import binding as B
N, d, V, R = 64, 64, 2000, 4
hid = torch.randn(N, d, device="cuda").bfloat16(); W = torch.randn(V, d, device="cuda").bfloat16()
off = torch.tensor(%s, dtype=torch.int32, device="cuda"); load = torch.zeros(R, device="cuda")
pr = B.Probe(N, d, V, R)
pr(hid, W, off, load, B.TauParams(l_target=0.5))
try:
    torch.cuda.synchronize()
except Exception as e:
    print("CUDA-ERROR", type(e).__name__); sys.exit(3)
print("OK", pr.exit.cpu().tolist())
"""
    env = dict(os.environ, LASER_DEBUG="1")
    good = subprocess.run([sys.executable, "-c", prog % (root, "[0, 16, 32, 48, 64]")], env=env,
                          capture_output=True, text=True, timeout=300)
    assert good.returncode == 0 and "OK" in good.stdout, good.stdout + good.stderr
    for bad_off in ("[0, 32, 16, 48, 64]", "[0, 16, 32, 48, 65]", "[1, 16, 32, 48, 64]"):
        bad = subprocess.run([sys.executable, "-c", prog % (root, bad_off)], env=env, capture_output=True,
                             text=True, timeout=300)
        assert bad.returncode != 0 and "OK" not in bad.stdout, (bad_off, bad.stdout, bad.stderr[-500:])
    # without LASER_DEBUG the same call is not checked (documented precondition) and must not trap
    env.pop("LASER_DEBUG")
    off_ok = subprocess.run([sys.executable, "-c", prog % (root, "[0, 16, 32, 48, 64]")], env=env,
                            capture_output=True, text=True, timeout=300)
    assert off_ok.returncode == 0


# ------------------------------------------------------------------------------- two real GPUs (skips on one)
def _two_gpu_worker(rank, world, port, exchange, q):
    import os
    import numpy as np
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dev = torch.device("cuda", rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    try:
        from paper_2606_31580_b200 import binding as B, parallel as par, workloads as wl
        w = wl.scaled("vp-2gpu", 9001, 256, 0.05, 40, None, seed=88, N_alloc=400, var_len=(1, 16))
        vp = par.VocabParallelProbe(dist, w.N_alloc, w.d, w.V, w.R, dev, exchange=exchange, debug_outputs=True)
        hidden = B.bf16_tensor_from_bits(w.hidden_bits, dev)
        Wg = B.bf16_tensor_from_bits(w.W_bits[vp.v0:vp.v1], dev)
        off = torch.from_numpy(w.req_offsets).to(dev)
        load = torch.from_numpy(w.load).to(dev)
        outs = []
        for it in range(6):          # several epochs: both peer buffer sets are reused
            out = vp(hidden, Wg, off, load, B.TauParams(**w.tau_params))
            torch.cuda.synchronize()
            outs.append([x.cpu().numpy().copy() for x in (out.conf, out.argmax, out.exit, out.tau, out.pmax)])
        q.put((rank, outs, vp.shard.plan))
    finally:
        dist.barrier()
        dist.destroy_process_group()


@pytest.mark.parametrize("exchange", ["peer", "collective"])
def test_vocab_parallel_two_gpus(P, exchange):
    """Cross-GPU run of the vocabulary-parallel probe: 2 ranks on 2 GPUs, records pushed over NVLink
    (peer) or all-gathered (collective); every rank's outputs against the oracle, six exchanges."""
    import socket
    import torch
    import torch.multiprocessing as mp
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (this pool leases one); the one-GPU virtual-rank tests cover the kernels")
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_two_gpu_worker, args=(r, 2, port, exchange, q)) for r in range(2)]
    for p_ in procs:
        p_.start()
    got = [q.get(timeout=600) for _ in procs]
    for p_ in procs:
        p_.join(timeout=60)
        assert p_.exitcode == 0
    w = wl.scaled("vp-2gpu", 9001, 256, 0.05, 40, None, seed=88, N_alloc=400, var_len=(1, 16))
    ora, rows, reqs = P.run_oracle(w)
    for rank, outs, plan in got:
        for it, o in enumerate(outs):
            P.compare(w, P.GpuRun(*o, plan), ora, rows, reqs, f"2gpu-{exchange}-rank{rank}-it{it}")
