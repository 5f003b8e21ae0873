"""-m gpu: the reusable plan (bqc_t_plan_*, include/bqc_t.h), the thread-local plan cache of bqc_t_energy_ex,
the memory budget option and the paper's largest shape."""
import os

import numpy as np
import pytest
import torch

import paper_2502_17963_b200 as bqc
from bqc_inputs import CONFIGS, make_config, make_inputs
from oracle import t_oracle as orc
from gpu_util import dims, e_tol, to_device

pytestmark = pytest.mark.gpu


def test_plan_is_reusable_across_inputs_and_matches_the_oracle():
    a = make_inputs(6, 18, 25, seed=5, t1_std=0.05, t2_std=0.03)
    b = make_inputs(6, 18, 25, seed=6, t1_std=0.05, t2_std=0.03)
    da, db = to_device(a), to_device(b)
    plan = bqc.bqc_t_plan(6, 18, 25, bqc.make_opts(occ_block=2, max_batch=3))
    assert plan.workspace_bytes() == bqc.bqc_t_workspace_bytes(6, 18, 25, bqc.make_opts(occ_block=2, max_batch=3))
    n = bqc.bqc_t_num_triplets(6)
    for inp, d in ((a, da), (b, db), (a, da)):
        et = torch.empty(n, dtype=torch.float64, device="cuda")
        e = plan.execute(*d, e_triplet=et)
        e_ref, trip_ref = orc.t_energy(inp, return_triplets=True)
        assert abs(e - e_ref) <= e_tol(e_ref)
        assert np.all(np.abs(et.cpu().numpy() - trip_ref) <= 1e-10 * np.abs(trip_ref) + 1e-12 * abs(e_ref) / n)
        # the one-shot call (which reuses its own cached plan) gives the same bits
        et2 = torch.empty_like(et)
        assert bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(occ_block=2, max_batch=3), e_triplet=et2) == e
        assert torch.equal(et, et2)
    plan.destroy()
    # a plan created without f_ov refuses one at execution, and vice versa
    plan = bqc.bqc_t_plan(6, 18, 25)
    f = torch.zeros((6, 18), dtype=torch.float64, device="cuda")
    with pytest.raises(bqc.BqcError) as ei:
        plan.execute(*da, f_ov=f)
    assert ei.value.code == 9
    plan.destroy()
    bqc.bqc_release_cached()


def test_fock_plan_and_f_ov_validation():
    inp = make_inputs(5, 12, 17, seed=9, t1_std=0.05, t2_std=0.03, f_std=0.05)
    d = to_device(inp)
    f = torch.from_numpy(inp.f_ov).cuda()
    plan = bqc.bqc_t_plan(5, 12, 17, bqc.make_opts(f_ov=f))
    e = plan.execute(*d, f_ov=f)
    e_ref = orc.t_energy(inp)
    assert abs(e - e_ref) <= e_tol(e_ref)
    plan.destroy()
    # binding-side validation of opts.f_ov (shape and memory space), ADVICE r1
    with pytest.raises(ValueError):
        bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(f_ov=f[:, :11].contiguous()))
    with pytest.raises(ValueError):
        bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(f_ov=f.cpu()))


def test_memory_budget_lowers_the_block_size_and_keeps_the_bits():
    inp = make_inputs(9, 40, 37, seed=12, t1_std=0.02)
    d = to_device(inp)
    n = bqc.bqc_t_num_triplets(9)
    base = torch.empty(n, dtype=torch.float64, device="cuda")
    e = bqc.bqc_t_energy_ex(*dims(inp), *d, e_triplet=base)
    # host-side: a smaller budget gives a smaller block and a smaller workspace at config 5
    big = bqc.bqc_t_workspace_bytes(100, 380, 1680)
    small = bqc.bqc_t_workspace_bytes(100, 380, 1680, bqc.make_opts(workspace_gib=12))
    assert small < big
    assert (bqc.bqc_t_plan_occ_block(100, 380, 1680, bqc.make_opts(workspace_gib=12))
            < bqc.bqc_t_plan_occ_block(100, 380, 1680))
    # device-side: explicit small blocks (several block triples, pair blocks re-formed) give the same e_ijk bits
    for bo in (2, 4):
        et = torch.empty_like(base)
        assert bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(occ_block=bo), e_triplet=et) == e
        assert torch.equal(et, base)
    # abc-driven, blocked over the virtual index: per-virtual-triple values independent of the block size
    v = inp.nvir
    A = bqc.BQC_T_FLAG_ABC_DRIVEN
    ref = torch.empty(bqc.bqc_t_num_triplets(v), dtype=torch.float64, device="cuda")
    ea = bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(flags=A), e_triplet=ref)
    assert abs(ea - e) <= e_tol(e)
    for bo in (7, 16):
        et = torch.empty_like(ref)
        assert bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(flags=A, occ_block=bo), e_triplet=et) == ea
        assert torch.equal(et, ref)


def _host_ram_gb():
    try:
        with open("/proc/meminfo") as fh:
            for ln in fh:
                if ln.startswith("MemAvailable:"):
                    return int(ln.split()[1]) / 1e6
    except OSError:
        pass
    return 0.0


def test_largest_shape_of_the_paper_runs_within_one_b200():
    """"capable of handling up to 1 380 orbitals".  Config 9 = (o, v, X) = (60, 1320, 4830), 117 GB
    of inputs: the abc-driven schedule on a window of 24 virtual orbitals, every array at full size.  The
    workspace stays far below the card (nothing of size o v^3 or v^2 o^2 is stored), and sampled per-virtual-
    triple values match the oracle's abc loop."""
    c = CONFIGS[9]
    o, v, X = c["nocc"], c["nvir"], c["naux"]
    A = bqc.BQC_T_FLAG_ABC_DRIVEN
    assert bqc.bqc_t_workspace_bytes(o, v, X, bqc.make_opts(flags=A)) < 45e9          # the full run
    opts = bqc.make_opts(occ_lo=40, occ_hi=64, flags=A)
    ws_bytes = bqc.bqc_t_workspace_bytes(o, v, X, opts)
    assert 0 < ws_bytes < 30e9
    free, total = torch.cuda.mem_get_info()
    if _host_ram_gb() < 150 or free < 150e9:
        pytest.skip("needs 150 GB of host memory and of device memory for the 117 GB input set")
    inp = make_config(9)
    d = [torch.from_numpy(a).cuda() for a in inp.arrays()]
    et = torch.empty(bqc.bqc_t_num_triplets(v), dtype=torch.float64, device="cuda")
    e = bqc.bqc_t_energy_ex(o, v, X, *d, opts=opts, e_triplet=et)
    ntr = 24 * 25 * 26 // 6 - 24
    idx = [bqc.bqc_t_triplet_index(v, a, b, cc) for (a, b, cc) in [(40, 41, 63), (45, 45, 50), (40, 63, 63), (47, 52, 60)]]
    got = et[torch.tensor(idx, device="cuda")].cpu().numpy()
    assert int(torch.count_nonzero(et)) == ntr
    del d, et
    torch.cuda.empty_cache()
    for g, (a, b, cc) in zip(got, [(40, 41, 63), (45, 45, 50), (40, 63, 63), (47, 52, 60)]):
        ref = orc.e_virtual_triple(inp, a, b, cc)
        assert abs(g - ref) <= 1e-10 * abs(ref) + 1e-12 * abs(e) / ntr, (a, b, cc, g, ref)
    bqc.bqc_release_cached()


def test_graph_replay_of_short_schedules_matches_the_eager_path():
    """Short schedules without BQC_T_FLAG_PROFILE are captured into a CUDA graph and replayed when the argument
    pointers repeat (the launch-bound regime).  Replays must track the VALUES behind the pointers,
    re-capture when a pointer changes, and give the same bits as the eager (profiled) path."""
    inp = make_config(1, t1_std=0.05)
    d = to_device(inp)
    n = bqc.bqc_t_num_triplets(inp.nocc)
    et = torch.empty(n, dtype=torch.float64, device="cuda")
    eager = torch.empty_like(et)
    e_eager = bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(flags=bqc.BQC_T_FLAG_PROFILE), e_triplet=eager)
    e_ref = orc.t_energy(inp)
    assert abs(e_eager - e_ref) <= e_tol(e_ref)
    for _ in range(3):                                   # capture, then two replays
        et.zero_()
        assert bqc.bqc_t_energy_ex(*dims(inp), *d, e_triplet=et) == e_eager
        assert torch.equal(et, eager)
    # new values behind the same pointers: the replay recomputes everything
    other = make_config(1, t1_std=0.05, seed=4242)
    for dst, src in zip(d, to_device(other)):
        dst.copy_(src)
    e2 = bqc.bqc_t_energy_ex(*dims(inp), *d, e_triplet=et)
    e2_ref = orc.t_energy(other)
    assert abs(e2 - e2_ref) <= e_tol(e2_ref) and e2 != e_eager
    # a different output pointer (and none at all): re-capture, same result
    et2 = torch.empty_like(et)
    assert bqc.bqc_t_energy_ex(*dims(inp), *d, e_triplet=et2) == e2 and torch.equal(et, et2)
    assert bqc.bqc_t_energy_ex(*dims(inp), *d) == e2
    assert bqc.bqc_t_energy(*dims(inp), *d) == e2
    # a vanishing denominator is still reported (the verdict travels with the result)
    d[1][0] = -2.0
    with pytest.raises(bqc.BqcError) as ei:
        bqc.bqc_t_energy_ex(*dims(inp), *d)
    assert ei.value.code == 8
    bqc.bqc_release_cached()
