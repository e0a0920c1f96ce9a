"""necsim_merge_species_static: the species-table merge with the library's static device scratch (no workspace, no allocation)
gives exactly what necsim_merge_species gives with a caller workspace. Collected last on purpose (the suite runs with -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _tables(idx, world):
    """Concatenated species tables of `world` isolated partitions of small config `idx` (duplicates across partitions included)."""
    import torch
    from paper_2108_05815_b200 import inputs as I, necsim as ns, dist as D
    cfg = I.small_configs()[idx]
    sc = ns.Scenario(**I.scenario_kwargs(cfg))
    tabs = []
    for r in range(world):
        m = D.shard_mask(cfg["mask"], sc.n_individuals, r, world)
        res = sc.simulate_raw(cfg["seed"], cfg["nu"], torch.from_numpy(m).cuda(), int(m.sum()), None)
        t, _ = sc.result_tensors(res)
        tabs.append(t.clone())
    sc.close()
    return torch.cat(tabs).contiguous()


def test_static_merge_equals_workspace_merge_two_calls_in_a_row():
    import torch
    from paper_2108_05815_b200 import necsim as ns
    big, small = _tables(1, 5), _tables(3, 2)            # the second call is the smaller one: it runs over the first call's leftovers
    assert big.numel() // 32 > small.numel() // 32 > 0
    for d_in in (big, small, big):
        n = d_in.numel() // 32
        want_tab, want_map = ns.merge_species(d_in)
        out = torch.full((n * 32,), 0xA5, dtype=torch.uint8, device="cuda")      # caller-owned outputs, poisoned
        dmap = torch.full((n,), -7, dtype=torch.int32, device="cuda")
        got_tab, got_map = ns.merge_species_static(d_in, out, dmap)
        torch.cuda.synchronize()
        assert got_tab.numel() == want_tab.numel() and got_tab.numel() > 0
        assert torch.equal(got_tab, want_tab)                                    # bit-exact: integer work
        assert torch.equal(got_map.to(torch.int64), want_map)
        ev = got_tab.cpu().numpy().view(ns.EVENT_DTYPE)
        assert int(ev["abundance"].sum()) == int(d_in.cpu().numpy().view(ns.EVENT_DTYPE)["abundance"].sum())


def test_static_merge_rejects_sizes_beyond_the_maximum():
    import torch
    from paper_2108_05815_b200 import necsim as ns
    n = ns.MERGE_STATIC_MAX + 1
    d_in = torch.zeros(n * 32, dtype=torch.uint8, device="cuda")
    with pytest.raises(ns.NecsimError) as e:
        ns.merge_species_static(d_in)
    assert "NECSIM_MERGE_STATIC_MAX" in str(e.value)
    # the maximum itself is accepted (records that are all equal: one species)
    d_in = torch.zeros(ns.MERGE_STATIC_MAX * 32, dtype=torch.uint8, device="cuda")
    tab, dmap = ns.merge_species_static(d_in)
    assert tab.numel() == 32 and int(dmap.max()) == 0
