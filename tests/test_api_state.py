"""Call-order cases of the C ABI: an entry point that leaves forces, lists or host buffers in a state the next call
misreads.  Each case compares a simulation that took the detour with a twin that did not, bit for bit."""
import pytest

import paper_1412_8502_b200 as pasta

pytestmark = pytest.mark.gpu


def _twin_steps(make, detour, steps=3, dt=2.0):
    """x, v after `steps` steps with and without `detour(sim)` before them."""
    import torch

    out = []
    for take in (False, True):
        with make() as sim:
            sim.energy()  # forces and energies are cached from here on
            if take:
                detour(sim)
            ke, pe = sim.energy()
            e = sim.particle_energies().clone()
            sim.step(steps, dt)
            x, v, _, _, _ = sim.get_state()
            torch.cuda.synchronize()
            out.append((x.clone(), v.clone(), e, ke, pe))
    return out


def test_force_stats_then_step_with_coulomb_all_pairs():
    """pasta_force_stats runs the chunk kernel alone; with coulomb_all_pairs its F lacks the whole Coulomb sum and must
    not be taken for the forces of the configuration (pasta_api.cu force_stats)."""
    import torch

    make = lambda: pasta.Sim(6000, 0.4, 0.003, 0.5, seed=9,  # noqa: E731
                             params=pasta.default_params(r_c=20.0, r_nuc=11.5, coulomb_all_pairs=1))
    (x0, v0, e0, ke0, pe0), (x1, v1, e1, ke1, pe1) = _twin_steps(make, lambda sim: sim.force_stats())
    assert pe1 == pe0 and ke1 == ke0 and torch.equal(e1, e0)
    assert torch.equal(x1, x0) and torch.equal(v1, v0)


def test_force_stats_then_step_when_sharded():
    """Under pasta_set_shard the statistics pass covers every target and issues no collective; what it leaves in F is the
    complete force on every rank, so the step that follows equals the unsharded one."""
    import torch

    make = lambda: pasta.Sim(6000, 0.3, 0.05, 0.5, seed=9, params=pasta.default_params(r_c=17.0))  # noqa: E731
    calls = []

    def detour(sim):
        sim.set_shard(1, 2, allreduce=lambda t: calls.append(t.numel()))  # forces become stale; the window is rank 1's
        sim.force_stats()
        n = len(calls)
        sim.set_shard(0, 1)      # NB marks forces stale again ...
        assert len(calls) == n == 0

    (x0, v0, e0, ke0, pe0), (x1, v1, e1, ke1, pe1) = _twin_steps(make, detour)
    assert pe1 == pe0 and torch.equal(e1, e0) and torch.equal(x1, x0) and torch.equal(v1, v0)
    # ... so look at F itself right after the statistics pass, still in sharded mode, without another evaluation
    with make() as sim:
        F_ref, _ = sim.forces()
        F_ref = F_ref.clone()
        sim.set_shard(1, 2, allreduce=lambda t: calls.append(t.numel()))
        sim.force_stats()
        x = torch.empty((sim.N, 3), dtype=torch.float64)
        F = torch.empty((sim.N, 3), dtype=torch.float64)
        sim.get_state_host(x=x, F=F)   # F is copied out as cached: no evaluation, hence no collective
        assert calls == []
        assert torch.equal(F.cuda(), F_ref)


def test_host_buffers_of_an_async_set_are_free_after_the_next_but_one():
    """pasta.h: the host buffers of pasta_set_state_host_async may be refilled once the next-but-one async set has
    returned.  The device is kept busy so that the uploads queue up behind it; the buffers of set 2 are overwritten the
    moment set 4 returns, and the state set 2 delivered must still be the original one."""
    import torch

    N = 20000
    with pasta.Sim(N, 0.3, 0.05, 0.5, seed=4, params=pasta.default_params(r_c=17.0)) as sim:
        L = sim.box_length()
        g = torch.Generator().manual_seed(1)
        xs = [(torch.rand((N, 3), generator=g, dtype=torch.float64) * (0.999 * L)).pin_memory() for _ in range(5)]
        vs = [(torch.randn((N, 3), generator=g, dtype=torch.float64) * 0.01).pin_memory() for _ in range(5)]
        keep = [(x.clone(), v.clone()) for x, v in zip(xs, vs)]
        rx = [torch.empty((N, 3), dtype=torch.float64).pin_memory() for _ in range(5)]
        rv = [torch.empty((N, 3), dtype=torch.float64).pin_memory() for _ in range(5)]
        sim.step(400, 2.0)                 # tens of milliseconds of queued work ahead of every take-over
        for k in range(5):
            sim.set_state_host_async(xs[k], vs[k])
            sim.get_state_host_async(rx[k], rv[k])
            if k >= 2:                     # set k has returned: the buffers of set k - 2 are the caller's again
                xs[k - 2].fill_(-1.0e9)
                vs[k - 2].fill_(7.0)
        sim.host_sync()
        for k in range(5):
            assert torch.equal(rx[k], keep[k][0]) and torch.equal(rv[k], keep[k][1]), "state of set %d was lost" % k


def test_cells_then_step_on_reused_lists_with_coulomb_all_pairs():
    """pasta_cells overwrites the cell-list scratch; reused neighbour lists must not outlive that (with coulomb_all_pairs
    the next evaluation used to stop with PASTA_ESTATE because the all-pairs kernel found no sorted protons)."""
    prm = dict(r_c=20.0, r_nuc=11.5, coulomb_all_pairs=1)
    res = []
    for detour in (False, True):
        with pasta.Sim(5000, 0.4, 0.0028, 0.5, seed=3, params=pasta.default_params(**prm)) as sim:
            sim.step(4, 2.0)
            st = sim.list_stats()
            assert st["list_builds"] < st["force_evals"]  # the neighbour-list regime, lists being reused
            if detour:
                cid, start, nc = sim.cells()
                assert int(start[-1]) == sim.N
            sim.step(4, 2.0)
            ke, pe = sim.energy()
            x = sim.get_state()[0].clone()
            res.append((ke, pe, x))
    (ke0, pe0, x0), (ke1, pe1, x1) = res
    # the detour costs a rebuild -- another sorted order, hence another FP32 summation order in the 4 steps that follow
    # (the gates test_neighbour_list_run_equals_run_without_it holds a run with lists to against one without) -- nothing else
    assert abs(pe1 - pe0) <= 1e-5 * abs(pe0) and abs(ke1 - ke0) <= 1e-5 * abs(ke0)
    assert float((x1 - x0).abs().max()) <= 1e-4


def test_lists_come_back_after_a_state_that_was_too_dense_for_them():
    """A list build that finds the state too dense switches lists off; a new state (pasta_set_state) or box (pasta_expand)
    must switch them on again."""
    import torch

    N, density = 12000, 0.001
    with pasta.Sim(N, 0.3, density, 0.5, seed=6, params=pasta.default_params(r_c=20.0)) as sim:
        x0, v0, _, L, _ = sim.get_state()
        x0, v0 = x0.clone(), v0.clone()

        def builds_over(n):
            a = sim.list_stats()
            for _ in range(n):
                sim.forces(want_pe=False)
            b = sim.list_stats()
            assert b["force_evals"] - a["force_evals"] == n
            return b["list_builds"] - a["list_builds"]

        assert builds_over(3) <= 1                      # dilute and uniform: built once (or already), then reused
        g = torch.Generator().manual_seed(2)
        # everything inside ONE row of the lists' grid (cells about 6.7 fm wide: floor(3 L / r_c) per side): a rod 50 fm
        # long and 5 fm thick through the middle of a cell -- more slots in one row stretch than a list record can count
        ncell = int(3.0 * L / 20.0)
        centre = (ncell // 2 + 0.5) * (L / ncell)
        lump = torch.rand((N, 3), generator=g, dtype=torch.float64) - 0.5
        lump = centre + lump * torch.tensor([50.0, 5.0, 5.0], dtype=torch.float64)
        sim.set_state(lump, torch.zeros_like(lump))
        assert builds_over(3) == 3                      # too dense for lists: the chunk path, a sort per evaluation
        sim.set_state(x0, v0)
        assert builds_over(3) == 1                      # lists again
        sim.set_state(lump, torch.zeros_like(lump))
        assert builds_over(2) == 2
        sim.expand(1.0)                                 # same lump, but the caller asked for a fresh start ...
        assert builds_over(2) == 2                      # ... lists are tried, found too dense again, and stay off
        sim.set_state(x0, v0)
        assert builds_over(3) == 1
