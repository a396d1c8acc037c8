"""The no-allocation entry point pswf_lr_exclusive_scan_static (include/pswf_lr.h): the cell-start scan of
step a0 with its scratch in a static device array of the library.  Collected last on purpose (the suite
runs with pytest -x: a failure here must not hide the other tests).

Integer work: compared BIT-EXACTLY with the existing path -- the cell starts a plan's evaluation leaves
behind (k_bin_count + the same scan kernel on the plan's cudaMalloc'd state), fetched with
pswf_lr_debug_cell_starts; the input of the new call is their first difference (the counts)."""
import numpy as np
import pytest
import torch

from paper_2606_06617_b200 import binding

pytestmark = pytest.mark.gpu


def _cell_starts_existing_path(grid, box, n_atoms, seed):
    """Cell starts int32[Mtot + 1] of one evaluation through the plan (the existing path), on the device."""
    rng = np.random.default_rng(seed)
    dev = torch.device("cuda:0")
    pos = torch.as_tensor(rng.uniform(0, 1, (n_atoms, 3)) * np.asarray(box), dtype=torch.float32, device=dev)
    q = torch.as_tensor(rng.normal(0, 0.5, (1, n_atoms)), dtype=torch.float32, device=dev)
    plan = binding.Plan(box, grid, 8, 12.024, [1])
    E = torch.zeros(1, dtype=torch.float64, device=dev)
    st = torch.cuda.current_stream().cuda_stream
    plan.execute(n_atoms, pos, q, E, None, None, st)
    starts = torch.empty(int(np.prod(grid)) + 1, dtype=torch.int32, device=dev)
    plan.debug_cell_starts(starts, st)
    torch.cuda.synchronize()
    plan.destroy()
    return starts


def test_static_scan_matches_plan_path_two_calls_in_a_row():
    # 40 x 48 x 56 = 107,520 cells: six full tiles of 16,384 counts and a ragged seventh;
    # 64^3 = 262,144 cells: sixteen full tiles.  Different inputs, so stale scratch would show.
    cases = [([40, 48, 56], [50.0, 60.0, 70.0], 30000, 11), ([64, 64, 64], [80.0, 80.0, 80.0], 50000, 12)]
    refs = [_cell_starts_existing_path(*c) for c in cases]
    bufs = []
    for ref in refs:
        counts = torch.empty_like(ref)
        counts[:-1] = ref[1:] - ref[:-1]
        counts[-1] = -12345                      # ignored on entry, receives the total
        assert int(counts[:-1].min()) >= 0 and int(counts[:-1].sum()) == int(ref[-1])
        bufs.append(counts)
    st = torch.cuda.current_stream().cuda_stream
    binding.exclusive_scan_static(bufs[0], bufs[0].numel() - 1, st)      # first call: resolves the symbol address
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    binding.exclusive_scan_static(bufs[1], bufs[1].numel() - 1, st)      # second call, right behind
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the device's free memory"
    for got, ref, c in zip(bufs, refs, cases):
        assert torch.equal(got, ref), "static-scratch scan differs from the plan's cell starts at grid %s" % c[0]
        assert int(got[-1]) == c[2]
    # and against the definition
    again = torch.empty_like(refs[0])
    cnt = (refs[0][1:] - refs[0][:-1]).to(torch.int64)
    again[:-1] = refs[0][1:] - refs[0][:-1]
    again[-1] = 7
    binding.exclusive_scan_static(again, again.numel() - 1, st)
    torch.cuda.synchronize()
    expect = torch.zeros(again.numel(), dtype=torch.int64, device=again.device)
    expect[1:] = torch.cumsum(cnt, 0)
    assert torch.equal(again.to(torch.int64), expect)


def test_static_scan_edges_and_limits():
    dev = torch.device("cuda:0")
    st = torch.cuda.current_stream().cuda_stream
    one = torch.tensor([5, -1, 0, 0], dtype=torch.int32, device=dev)
    binding.exclusive_scan_static(one, 1, st)
    empty = torch.tensor([9, 9, 9, 9], dtype=torch.int32, device=dev)
    binding.exclusive_scan_static(empty, 0, st)
    torch.cuda.synchronize()
    assert one[:2].tolist() == [0, 5]
    assert empty.tolist() == [0, 9, 9, 9]
    small = torch.zeros(8, dtype=torch.int32, device=dev)
    with pytest.raises(binding.PswfLrError) as e:                        # rejected before anything is touched
        binding.exclusive_scan_static(small, binding.SCAN_STATIC_MAX + 1, st)
    assert e.value.code == binding.ERR_TOO_LARGE
    with pytest.raises(binding.PswfLrError) as e:
        binding.exclusive_scan_static(small, -1, st)
    assert e.value.code == binding.ERR_INVALID_ARG
    with pytest.raises(binding.PswfLrError) as e:
        binding.exclusive_scan_static(small[1:], 4, st)                  # not 16-byte aligned
    assert e.value.code == binding.ERR_INVALID_ARG
    with pytest.raises(binding.PswfLrError) as e:
        binding.exclusive_scan_static(None, 4, st)
    assert e.value.code == binding.ERR_INVALID_ARG
    # the full maximum: 2^24 counts of 1 -> starts 0, 1, 2, ...
    big = torch.ones(binding.SCAN_STATIC_MAX + 1, dtype=torch.int32, device=dev)
    binding.exclusive_scan_static(big, binding.SCAN_STATIC_MAX, st)
    torch.cuda.synchronize()
    assert torch.equal(big, torch.arange(binding.SCAN_STATIC_MAX + 1, dtype=torch.int32, device=dev))
