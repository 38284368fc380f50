"""ising_energy_cut_noalloc (include/ising_noalloc.h): the entry point that allocates nothing (static device scratch)
against the existing ising_energy_cut path, two calls in a row.  Integers: bit-exact.  Collected last on purpose."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _device_csr(wl, torch):
    return (torch.from_numpy(np.ascontiguousarray(wl.row_ptr, dtype=np.int64)).cuda(),
            torch.from_numpy(np.ascontiguousarray(wl.col, dtype=np.int32)).cuda(),
            torch.from_numpy(np.ascontiguousarray(wl.w)).cuda())


def test_noalloc_energy_cut_matches_existing_path_twice():
    import torch
    import paper_1807_10750_b200 as P
    from paper_1807_10750_b200 import binding as B, workloads as W

    rng = np.random.default_rng(20260511)
    # two different graphs / replica counts back to back: the second call must not see the first one's scratch
    cases = [W.config5(n=3000, sweeps=1, replicas=37),      # int8 weights, hubs, a ragged replica count
             W.config1(sweeps=1)]                           # int32 weights, 1 replica
    for rounds in range(2):
        for wl in cases:
            R = wl.n_replicas
            spins = (rng.integers(0, 2, size=(R, wl.n), dtype=np.int8) * 2 - 1).astype(np.int8)
            p = P.load_workload(wl)
            e_ref, c_ref = P.ising_energy_cut(p, spins)                     # existing path (handle + workspace)
            row_ptr, col, w = _device_csr(wl, torch)
            d_spins = torch.from_numpy(spins).cuda()
            e = torch.full((R,), -7, dtype=torch.int64, device="cuda")
            c = torch.full((R,), -7, dtype=torch.int64, device="cuda")
            torch.cuda.synchronize()
            B.ising_energy_cut_noalloc(row_ptr, col, w, d_spins, e, c)     # first call
            e1, c1 = e.clone(), c.clone()
            e.fill_(-7); c.fill_(-7)
            B.ising_energy_cut_noalloc(row_ptr, col, w, d_spins, e, c)     # second call in a row: same scratch
            torch.cuda.synchronize()
            np.testing.assert_array_equal(e1.cpu().numpy(), e_ref.cpu().numpy())
            np.testing.assert_array_equal(c1.cpu().numpy(), c_ref.cpu().numpy())
            np.testing.assert_array_equal(e.cpu().numpy(), e_ref.cpu().numpy())
            np.testing.assert_array_equal(c.cpu().numpy(), c_ref.cpu().numpy())
            # independent of the library: the definition in numpy (cut = weight of the edges whose endpoints differ)
            r0 = np.repeat(np.arange(wl.n), np.diff(wl.row_ptr))
            differ = spins[:, r0] != spins[:, wl.col]
            cut_np = (differ * wl.w.astype(np.int64)[None, :]).sum(axis=1) // 2
            np.testing.assert_array_equal(c.cpu().numpy(), cut_np)
            p.free()


def test_noalloc_rejects_sizes_beyond_the_scratch():
    import torch
    from paper_1807_10750_b200 import binding as B, workloads as W

    wl = W.config1(sweeps=1)
    row_ptr, col, w = _device_csr(wl, torch)
    R = B.NOALLOC_MAX_REPLICAS + 1
    spins = torch.ones((R, wl.n), dtype=torch.int8, device="cuda")
    e = torch.zeros(R, dtype=torch.int64, device="cuda")
    with pytest.raises(B.IsingError) as ei:
        B.ising_energy_cut_noalloc(row_ptr, col, w, spins, e, None)
    assert "replica" in str(ei.value).lower()
    # the largest size that fits works, cut only
    R = B.NOALLOC_MAX_REPLICAS
    c = torch.zeros(R, dtype=torch.int64, device="cuda")
    B.ising_energy_cut_noalloc(row_ptr, col, w, spins[:R].contiguous(), None, c)
    torch.cuda.synchronize()
    assert int(c.min()) == 0 and int(c.max()) == 0      # all spins equal: nothing is cut
