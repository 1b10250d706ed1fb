"""GPU parity of the intra-mesh sharding: one mesh cut into 2 / 3 parts, every part its own handle on
this device, one halo exchange per step (ep_halo_exchange_local), merged result against the oracle on the WHOLE mesh and
against the unsharded GPU run.  On several GPUs the exchange is the same pack / unpack with NCCL send/recv of the buffers
(ep_shard_buffers) in between; the lists themselves are checked across processes in tests/test_shard_plan.py."""
import numpy as np
import pytest

from ep_inputs import make, states

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ep():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2112_12854_b200 as ep
    return ep


def _shards(ep, prob, n_parts):
    m = prob.mesh
    sims = []
    for p in range(n_parts):
        s = ep.Sim.shard(m.xyz, m.tets, p, n_parts, m.fibre, m.sigma_scale, prob.sigma_l, prob.sigma_t, prob.chi, prob.Cm)
        ct = None if m.cell_type is None else m.cell_type[s.global_ids]
        s.state_init(prob.model, ct)
        loc = {int(g): k for k, g in enumerate(s.global_ids)}
        for k, st in enumerate(prob.stimuli):
            ids = np.array([loc[int(c)] for c in st.cell_ids if int(c) in loc], dtype=np.int64)
            s.stimulus_set(k, ids, st.amplitude, st.t_start, st.duration)
        sims.append(s)
    return sims


def _merge(sims, n, read):
    out = np.full(n, np.nan)
    for s in sims:
        out[s.global_ids[: s.n_owned]] = read(s)[: s.n_owned]
    assert not np.isnan(out).any()
    return out


@pytest.mark.parametrize("cfg,coarsen,n_parts", [(1, 1.0, 2), (1, 1.0, 3), (3, 4.0, 2)])
def test_sharded_run_equals_the_whole_mesh(ep, oracle, cfg, coarsen, n_parts, capsys):
    prob = make(cfg, coarsen=coarsen)
    n = prob.mesh.n_tets
    sims = _shards(ep, prob, n_parts)
    whole = ep.Sim.from_problem(prob)
    oracle.set_threads(8)
    o = oracle.OracleSim.from_problem(prob)
    dt = prob.dt
    steps = 300
    for _ in range(steps):
        for s in sims:
            s.step(1, dt)
        ep.halo_exchange_local(sims)
    whole.step(steps, dt)
    o.step(steps, dt)
    v = _merge(sims, n, lambda s: s.read_vm())
    ta = _merge(sims, n, lambda s: s.activation_times())
    dv_o = np.abs(v - o.read_vm()).max()
    dv_w = np.abs(v - whole.read_vm()).max()
    halo = sum(s.n_tets - s.n_owned for s in sims)
    with capsys.disabled():
        print("config %d (%d cells) in %d parts, %d halo cells, %d steps: max|dVm| vs oracle %.3e mV, vs unsharded GPU run %.3e mV"
              % (cfg, n, n_parts, halo, steps, dv_o, dv_w))
    assert dv_o <= 1e-6 and dv_w <= 1e-9
    ta_o = o.activation_times()
    assert np.array_equal(ta >= 0, ta_o >= 0) and (ta >= 0).sum() > 0 and np.abs(ta - ta_o).max() <= dt + 1e-12
    for k in (1, 9, 16):
        a = _merge(sims, n, lambda s: s.read_state(k))
        assert np.abs(a - o.read_state(k)).max() <= 1e-8 * max(1.0, np.abs(o.read_state(k)).max())
    # volume-weighted mean of the parts' means = the global mean
    vb = whole.mean_vm()
    parts = [(s.mean_vm(), s) for s in sims]
    # weights: owned volume of each part = its share of the cells on these equal-volume lattices only for config 1
    if cfg == 1:
        w = np.array([s.n_owned for _, s in parts], dtype=float)
        assert abs((w * np.array([m_ for m_, _ in parts])).sum() / w.sum() - vb) <= 1e-9
    for s in sims:
        assert s.check_finite()
        s.close()
    whole.close(); o.close()


def test_one_step_from_random_states_sharded(ep, oracle):
    prob = make(3, coarsen=4.0)
    n = prob.mesh.n_tets
    sims = _shards(ep, prob, 2)
    o = oracle.OracleSim.from_problem(prob)
    y = states.random_states(0, 61, n)
    for k in range(19):
        o.write_state(k, y[k])
        for s in sims:
            s.write_state(k, y[k][s.global_ids])
    for s in sims:
        s.step(1, 0.01)
    ep.halo_exchange_local(sims)
    o.step(1, 0.01)
    for k in range(19):
        a = _merge(sims, n, lambda s: s.read_state(k))
        b = o.read_state(k)
        assert np.abs(a - b).max() <= 1e-11 * np.abs(b).max(), k
    # after the exchange the halo copies equal the owners' values
    v = _merge(sims, n, lambda s: s.read_vm())
    for s in sims:
        assert np.array_equal(s.read_vm(), v[s.global_ids])
        s.close()
    o.close()


def test_shard_errors(ep):
    prob = make(1)
    m = prob.mesh
    whole = ep.Sim.from_problem(prob)
    with pytest.raises(ep.EpError):
        whole.halo_pack()                       # not a shard
    a = ep.Sim.shard(m.xyz, m.tets, 0, 2)
    b = ep.Sim.shard(m.xyz, m.tets, 1, 2)
    with pytest.raises(ep.EpError):
        ep.halo_exchange_local([b, a])          # wrong order
    for s in (whole, a, b):
        s.close()
