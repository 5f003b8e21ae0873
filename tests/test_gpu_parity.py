"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerances: energies |dE| <= 1e-10 |E| + 1e-12 Eh (BASELINE.json north_star); intermediates
(slabs, W, V) |d| <= 1e-11 * max|x| — FP64 sums of <= 6(v+o)+naux products in a different order
than the oracle's BLAS.
"""
import numpy as np
import pytest
import torch

import paper_2502_17963_b200 as bqc
from bqc_inputs import make_config, make_inputs, sample_triplets, worked_example
from gpu_util import dims, e_tol, to_device
from oracle import t_oracle as orc

pytestmark = pytest.mark.gpu


def _close(got, ref, rel=1e-11):
    got = got.cpu().numpy() if isinstance(got, torch.Tensor) else np.asarray(got)
    scale = np.max(np.abs(ref)) + 1e-300
    err = np.max(np.abs(got - ref))
    assert err <= rel * scale, f"max err {err:.3e} vs scale {scale:.3e}"


# ------------------------------------------------------------------ the tile-GEMM engine alone
@pytest.mark.parametrize("M,N,K", [(128, 128, 16), (1, 1, 1), (130, 70, 37), (517, 261, 100), (64, 300, 480),
                                   (1000, 19, 24)])
def test_dgemm_nt(M, N, K):
    rng = np.random.default_rng(M * 7 + N * 3 + K)
    lda = K + (K % 2) + 2
    A = np.zeros((M, lda)); A[:, :K] = rng.normal(size=(M, K))
    B = np.zeros((N, lda)); B[:, :K] = rng.normal(size=(N, K))
    A[:, K:] = 7.0   # stride padding must never be read as data
    B[:, K:] = -3.0
    dA = torch.from_numpy(A).cuda()[:, :K]
    dB = torch.from_numpy(B).cuda()[:, :K]
    C = bqc.bqc_dgemm_nt(dA, dB)
    _close(C, A[:, :K] @ B[:, :K].T, rel=1e-13 * max(K, 16))


# ------------------------------------------------------------------ row a1: DF slabs
@pytest.mark.parametrize("case", ["config1", "odd", "config2"])
def test_df_slabs(case):
    inp = {"config1": lambda: make_config(1), "odd": lambda: make_inputs(3, 21, 13, seed=5),
           "config2": lambda: make_config(2)}[case]()
    d = to_device(inp)
    o = inp.nocc
    for (x, y) in [(0, 0), (o - 1, 1), (1, o - 1)]:
        I, O, J = bqc.bqc_t_debug_slabs(*dims(inp), d[3], d[4], d[5], d[6], x, y)
        _close(I, orc.slab_vvov(inp, x))
        _close(O, orc.slab_ooov(inp, x, y))
        _close(J, orc.slab_ovov(inp, x, y))


# ------------------------------------------------------------------ rows a2 + a3: W and V
@pytest.mark.parametrize("case", ["worked346", "config1", "ragged", "twoseg", "config2"])
def test_w_and_v_elementwise(case):
    inp = {"worked346": lambda: worked_example(3, 4, 6), "config1": lambda: make_config(1),
           "ragged": lambda: make_inputs(4, 35, 41, seed=8, t1_std=0.05),
           "twoseg": lambda: make_inputs(3, 137, 21, seed=9, t1_std=0.05),   # N split into 5 + 4 groups of 16
           "config2": lambda: make_config(2, t1_std=0.05)}[case]()
    d = to_device(inp)
    o = inp.nocc
    trips = [(0, 1, 2), (0, 0, o - 1), (1, o - 1, o - 1), (2, 0, 1), (1, 1, 1)]
    if case == "config2":
        trips = [(3, 11, 19), (7, 7, 2)]
    for (i, j, k) in trips:
        W, V = bqc.bqc_t_debug_wv(*dims(inp), *d, i, j, k)
        Wr = orc.w_triplet(inp, i, j, k)
        _close(W, Wr)
        _close(V, orc.v_triplet(inp, i, j, k, Wr))


# ------------------------------------------------------------------ rows a4 + a5: energies
SMALL = {
    "worked234": lambda: worked_example(2, 3, 4),
    "worked346": lambda: worked_example(3, 4, 6),
    "config1": lambda: make_config(1),
    "config1_t1": lambda: make_config(1, t1_std=0.05),          # a3 exercised at O(1) weight
    "v16": lambda: make_inputs(3, 16, 10, seed=31, t1_std=0.05),  # exactly one 16-block
    "v17": lambda: make_inputs(4, 17, 9, seed=32, t1_std=0.05),   # ragged tail of 1
    "v33": lambda: make_inputs(3, 33, 20, seed=33, t1_std=0.05),  # 3 blocks, ragged
    "o2": lambda: make_inputs(2, 9, 5, seed=34, t1_std=0.05),
    "v1": lambda: make_inputs(3, 1, 4, seed=37, t1_std=0.05),       # a single virtual orbital
    "x1": lambda: make_inputs(3, 5, 1, seed=38, t1_std=0.05),       # a single auxiliary function
    "v137": lambda: make_inputs(3, 137, 24, seed=35, t1_std=0.05),  # 9 column groups: two GEMM column segments
    "v209": lambda: make_inputs(2, 209, 16, seed=36, t1_std=0.05),  # 14 groups = 7 + 7, ragged 8-block tail
}


@pytest.mark.parametrize("case", sorted(SMALL))
def test_energy_small_full(case):
    inp = SMALL[case]()
    d = to_device(inp)
    e_ref, trip_ref = orc.t_energy(inp, return_triplets=True)
    et = torch.empty(bqc.bqc_t_num_triplets(inp.nocc), dtype=torch.float64, device="cuda")
    e = bqc.bqc_t_energy_ex(*dims(inp), *d, e_triplet=et)
    assert abs(e - e_ref) <= e_tol(e_ref)
    got = et.cpu().numpy()
    n = len(trip_ref)
    # (1e-20 Eh floor: with a single virtual orbital every term cancels analytically and both sides return noise)
    assert np.all(np.abs(got - trip_ref) <= 1e-10 * np.abs(trip_ref) + 1e-12 * abs(e_ref) / n + 1e-20)
    # plain entry point
    assert bqc.bqc_t_energy(*dims(inp), *d) == e


def test_golden_worked_example_values():
    # SURVEY.md §8(c) P2 (tests/golden/worked_examples.txt)
    for shape, want in {(2, 3, 4): -9.406698159242249e-07, (3, 4, 6): -1.851157457841839e-04}.items():
        inp = worked_example(*shape)
        e = bqc.bqc_t_energy(*dims(inp), *to_device(inp))
        assert abs(e - want) <= e_tol(want)


def test_no_t1_flag_gives_e4():
    inp = make_config(1, t1_std=0.05)
    e4 = orc.t_energy(inp, with_t1=False)
    e = bqc.bqc_t_energy_ex(*dims(inp), *to_device(inp), opts=bqc.make_opts(flags=bqc.BQC_T_FLAG_NO_T1))
    assert abs(e - e4) <= e_tol(e4)


def test_single_occupied_is_exactly_zero():
    inp = make_inputs(1, 6, 8, seed=2, t1_std=0.05, t2_std=0.05)
    assert bqc.bqc_t_energy(*dims(inp), *to_device(inp)) == 0.0


def test_config2_full_energy_and_every_triplet():
    """the full oracle on config 2 — E(T) and all 1 540 per-triplet values."""
    inp = make_config(2)
    d = to_device(inp)
    o = inp.nocc
    et = torch.empty(bqc.bqc_t_num_triplets(o), dtype=torch.float64, device="cuda")
    e = bqc.bqc_t_energy_ex(*dims(inp), *d, e_triplet=et)
    got = et.cpu().numpy()
    e_ref, trip_ref = orc.t_energy(inp, return_triplets=True)
    assert len(trip_ref) == 1540
    assert abs(e - e_ref) <= e_tol(e_ref)
    assert np.all(np.abs(got - trip_ref) <= 1e-10 * np.abs(trip_ref) + 1e-12 * abs(e_ref) / 1540)
    assert bqc.bqc_t_energy(*dims(inp), *d) == e


def test_config3_sixteen_seeded_triplets():
    """a seeded subset of 16 triplets (seed 103) of config 3, plus any-size properties."""
    cfg, count = 3, 16
    inp = make_config(cfg)
    d = to_device(inp)
    o = inp.nocc
    et = torch.empty(bqc.bqc_t_num_triplets(o), dtype=torch.float64, device="cuda")
    e = bqc.bqc_t_energy_ex(*dims(inp), *d, e_triplet=et)
    got = et.cpu().numpy()
    assert abs(got.sum() - e) <= 1e-12 * abs(e)
    n = len(got)
    for (i, j, k) in sample_triplets(o, count, seed=100 + cfg):
        ref = orc.e_triplet(inp, i, j, k)
        g = got[bqc.bqc_t_triplet_index(o, i, j, k)]
        assert abs(g - ref) <= 1e-10 * abs(ref) + 1e-12 * abs(e) / n, (i, j, k, g, ref)
    # properties that hold at any size: diagonal triplets are exactly 0, E[4]-dominated values < 0
    for i in range(o):
        assert got[bqc.bqc_t_triplet_index(o, i, i, i)] == 0.0
    assert np.all(got <= 0.0)


@pytest.mark.parametrize("cfg", [4, 5])
def test_full_size_bench_configuration_sampled(cfg):
    """BASELINE.json configs[3], configs[4] at full array sizes, in the launch configuration
    bench.py times (occupied window [0,10), automatic slab block and batch): sampled per-triplet
    outputs (one i=j<k, one i<j=k, one i<j<k) against the oracle, plus the any-size properties."""
    inp = make_config(cfg)
    d = to_device(inp)
    o = inp.nocc
    opts = bqc.make_opts(occ_lo=0, occ_hi=10)
    et = torch.empty(bqc.bqc_t_num_triplets(o), dtype=torch.float64, device="cuda")
    e = bqc.bqc_t_energy_ex(*dims(inp), *d, opts=opts, e_triplet=et)
    got = et.cpu().numpy()
    assert abs(got.sum() - e) <= 1e-12 * abs(e)
    inside = 0
    for (i, j, k) in orc.triplet_list(10):
        idx = bqc.bqc_t_triplet_index(o, i, j, k)
        if i == j == k:
            assert got[idx] == 0.0
        else:
            assert got[idx] < 0.0
            inside += 1
    assert inside == 210 and np.count_nonzero(got) == 210        # nothing outside the window
    # eight triplets of the window: the three classes by hand + a seeded draw (seed 40 + cfg)
    rng = np.random.default_rng(40 + cfg)
    trips = [(2, 2, 7), (0, 9, 9), (1, 4, 8)]
    while len(trips) < 8:
        t = tuple(sorted(int(x) for x in rng.integers(0, 10, size=3)))
        if t not in trips and not (t[0] == t[1] == t[2]):
            trips.append(t)
    for (i, j, k) in trips:
        ref = orc.e_triplet(inp, i, j, k)
        g = got[bqc.bqc_t_triplet_index(o, i, j, k)]
        assert abs(g - ref) <= 1e-10 * abs(ref) + 1e-12 * abs(e) / 210, (i, j, k, g, ref)
    if cfg == 4:
        # one abc-driven sample at full size: a virtual window of 8, three virtual triples against the oracle's
        # separately written abc loop
        v = inp.nvir
        aopts = bqc.make_opts(occ_lo=0, occ_hi=8, flags=bqc.BQC_T_FLAG_ABC_DRIVEN)
        eta = torch.empty(bqc.bqc_t_num_triplets(v), dtype=torch.float64, device="cuda")
        ea = bqc.bqc_t_energy_ex(*dims(inp), *d, opts=aopts, e_triplet=eta)
        ga = eta.cpu().numpy()
        assert np.count_nonzero(ga) == 8 * 9 * 10 // 6 - 8
        for (a, b, c) in [(0, 3, 7), (2, 2, 5), (1, 6, 6)]:
            ref = orc.e_virtual_triple(inp, a, b, c)
            g = ga[bqc.bqc_t_triplet_index(v, a, b, c)]
            assert abs(g - ref) <= 1e-10 * abs(ref) + 1e-12 * abs(ea) / 112, (a, b, c, g, ref)
        del eta
    # single W / V elements straight from Eq. (2) (6 + 6 dot products), ragged tail included
    W, V = bqc.bqc_t_debug_wv(*dims(inp), *d, 1, 4, 8)
    v = inp.nvir
    scale = float(W.abs().max())
    for (a, b, c) in [(0, 0, 0), (v - 1, v - 1, v - 1), (17, v - 1, 130), (255, 16, v - 3)]:
        w_ref = orc.w_element(inp, 1, 4, 8, a, b, c)
        assert abs(float(W[a, b, c]) - w_ref) <= 1e-11 * scale
        assert abs(float(V[a, b, c]) - orc.v_element(inp, 1, 4, 8, a, b, c, w_ref)) <= 1e-11 * scale


# ------------------------------------------------------------------ scheduler: windows, blocks, shards
def test_blocking_window_and_sharding_agree_bitwise():
    inp = make_inputs(7, 20, 18, seed=41, t1_std=0.02)
    d = to_device(inp)
    n = bqc.bqc_t_num_triplets(7)
    base = torch.empty(n, dtype=torch.float64, device="cuda")
    e = bqc.bqc_t_energy_ex(*dims(inp), *d, e_triplet=base)
    assert abs(e - orc.t_energy(inp)) <= e_tol(e)
    for bo, mb in [(1, 1), (2, 3), (3, 0), (4, 2)]:
        et = torch.empty_like(base)
        e2 = bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(occ_block=bo, max_batch=mb), e_triplet=et)
        assert torch.equal(et, base), (bo, mb)     # same per-triplet arithmetic whatever the blocking
        assert e2 == e
    # shards: disjoint supports that add up to the whole
    parts = []
    for r in range(3):
        et = torch.empty_like(base)
        bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(shard_rank=r, shard_count=3, occ_block=3), e_triplet=et)
        parts.append(et)
    assert torch.equal(parts[0] + parts[1] + parts[2], base)
    for idx in range(n):
        assert sum(int(p[idx] != 0) for p in parts) <= 1
    # window: only triplets inside [2,6)
    et = torch.empty_like(base)
    ew = bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(occ_lo=2, occ_hi=6), e_triplet=et)
    ref = 0.0
    for (i, j, k) in orc.triplet_list(7):
        idx = bqc.bqc_t_triplet_index(7, i, j, k)
        if 2 <= i and k < 6:
            assert et[idx] == base[idx]
            ref += orc.e_triplet(inp, i, j, k)
        else:
            assert et[idx] == 0.0
    assert abs(ew - ref) <= e_tol(ref)


def test_block_triple_sharding_is_disjoint_bitwise_and_forms_fewer_slabs():
    """BQC_T_FLAG_SHARD_BLOCKS: whole block triples per shard."""
    inp = make_inputs(9, 19, 13, seed=53, t1_std=0.05)
    d = to_device(inp)
    o = inp.nocc
    n = bqc.bqc_t_num_triplets(o)
    base = torch.empty(n, dtype=torch.float64, device="cuda")
    e_all = bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(occ_block=2, flags=bqc.BQC_T_FLAG_PROFILE),
                                e_triplet=base)
    forms_all = bqc.bqc_t_last_profile()["form_blocks"]
    F = bqc.BQC_T_FLAG_SHARD_BLOCKS | bqc.BQC_T_FLAG_PROFILE
    for world in (2, 3, 5):
        parts, flops, forms, es = [], 0.0, [], []
        for r in range(world):
            et = torch.empty_like(base)
            opts = bqc.make_opts(shard_rank=r, shard_count=world, occ_block=2, flags=F)
            es.append(bqc.bqc_t_energy_ex(*dims(inp), *d, opts=opts, e_triplet=et))
            forms.append(bqc.bqc_t_last_profile()["form_blocks"])
            flops += bqc.bqc_t_flops(o, inp.nvir, opts)
            # the flop model counts exactly the triplets this shard evaluated
            nz = int((et != 0).sum())
            assert bqc.bqc_t_flops(o, inp.nvir, opts) == nz * 12.0 * inp.nvir ** 3 * (inp.nvir + o)
            parts.append(et)
        assert torch.equal(sum(parts), base)                                # same bits, every triplet once
        for idx in range(n):
            assert sum(int(p[idx] != 0) for p in parts) <= 1
        assert flops == bqc.bqc_t_flops(o, inp.nvir)
        assert abs(sum(es) - e_all) <= e_tol(e_all)
        assert max(forms) < forms_all                                       # a shard forms only what it needs
    # one shard: the flag changes nothing
    et = torch.empty_like(base)
    bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(occ_block=2, flags=bqc.BQC_T_FLAG_SHARD_BLOCKS), e_triplet=et)
    assert torch.equal(et, base)


def test_deterministic_and_workspace_and_host_paths():
    inp = make_config(1, t1_std=0.01)
    d = to_device(inp)
    e1 = bqc.bqc_t_energy(*dims(inp), *d)
    e2 = bqc.bqc_t_energy(*dims(inp), *d)
    assert e1 == e2                                             # bit-identical
    ws = torch.empty(bqc.bqc_t_workspace_bytes(*dims(inp)), dtype=torch.uint8, device="cuda")
    assert bqc.bqc_t_energy_ex(*dims(inp), *d, workspace=ws) == e1
    with pytest.raises(bqc.BqcError) as ei:
        bqc.bqc_t_energy_ex(*dims(inp), *d, workspace=ws[:1024])
    assert ei.value.code == 5
    host = [torch.from_numpy(a) for a in inp.arrays()]
    eh, h2d, d2h = bqc.bqc_t_energy_host(*dims(inp), *host)
    assert eh == e1 and h2d == inp.nbytes() and d2h == 8
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        assert bqc.bqc_t_energy(*dims(inp), *d) == e1           # non-default stream


def test_host_entry_point_with_a_window_copies_only_the_t2_rows_it_reads():
    inp = make_inputs(7, 18, 13, seed=52, t1_std=0.05)
    o, v, X = dims(inp)
    d = to_device(inp)
    host = [torch.from_numpy(np.ascontiguousarray(a)) for a in inp.arrays()]
    for lo, hi in [(0, 3), (2, 6), (4, 7)]:
        opts = bqc.make_opts(occ_lo=lo, occ_hi=hi)
        et_d = torch.zeros(bqc.bqc_t_num_triplets(o), dtype=torch.float64, device="cuda")
        e_dev = bqc.bqc_t_energy_ex(o, v, X, *d, opts=opts, e_triplet=et_d)
        et_h = torch.zeros(bqc.bqc_t_num_triplets(o), dtype=torch.float64)
        e_host, h2d, d2h = bqc.bqc_t_energy_host(o, v, X, *host, opts=opts, e_triplet=et_h)
        assert e_host == e_dev and np.array_equal(et_h.numpy(), et_d.cpu().numpy())     # same bits
        assert h2d == inp.nbytes() - inp.t2.nbytes + (hi - lo) * o * v * v * 8
        # and it is the oracle's value for those triplets
        ref = sum(orc.e_triplet(inp, i, j, k) for i in range(lo, hi) for j in range(i, hi) for k in range(j, hi))
        assert abs(e_host - ref) <= e_tol(ref)


# ------------------------------------------------------------------ error behaviour (no CPU fallback)
def test_errors_are_reported():
    inp = make_config(1)
    d = to_device(inp)
    o, v, x = dims(inp)
    L = bqc.lib()
    import ctypes
    ptrs = [ctypes.c_void_p(t.data_ptr()) for t in d]
    e = ctypes.c_double(0)
    def call(o_=o, v_=v, x_=x, p=ptrs):
        return L.bqc_t_energy_ex(o_, v_, x_, *p, None, None, 0, ctypes.byref(e), None, None)
    assert call(o_=0) == 1
    assert call(p=[None] + ptrs[1:]) == 2
    host = torch.from_numpy(inp.t2)
    assert call(p=ptrs[:3] + [ctypes.c_void_p(host.data_ptr())] + ptrs[4:]) == 3
    assert call(p=[ctypes.c_void_p(d[0].data_ptr() + 4)] + ptrs[1:]) == 4
    bad = d[0].clone(); bad[-1] = 1.0                            # occupied level above a virtual one
    assert call(p=[ctypes.c_void_p(bad.data_ptr())] + ptrs[1:]) == 8
    assert L.bqc_last_error() == 8 and b"denominator" in L.bqc_error_detail()
    import math
    assert math.isnan(L.bqc_t_energy(0, v, x, *ptrs, None))
    assert call() == 0                                           # and the library still works


# ------------------------------------------------------------------ NEXT-3: occupied-virtual Fock block
@pytest.mark.parametrize("case", ["o3v16", "config1", "ragged"])
def test_fock_term_energy_and_v(case):
    """PAPER.md:298-303 Eqs. (5),(7) (reading G15): V += f[i,a] t2[j,k,b,c] + f[j,b] t2[i,k,a,c] + f[k,c] t2[i,j,a,b]."""
    import copy
    inp = {"o3v16": lambda: make_inputs(3, 16, 10, seed=41, t1_std=0.05, f_std=0.1),
           "config1": lambda: make_config(1, t1_std=0.05, f_std=0.05),
           "ragged": lambda: make_inputs(4, 35, 41, seed=42, t1_std=0.05, f_std=0.1)}[case]()
    d = to_device(inp)
    f_dev = torch.from_numpy(inp.f_ov).cuda()
    e_ref, trip_ref = orc.t_energy(inp, return_triplets=True)
    canon = copy.copy(inp)
    canon.f_ov = None
    e_canon = orc.t_energy(canon)
    assert abs(e_ref - e_canon) > 1e-6 * abs(e_ref)          # the term carries weight in this input
    et = torch.empty(bqc.bqc_t_num_triplets(inp.nocc), dtype=torch.float64, device="cuda")
    e = bqc.bqc_t_energy_ex(*dims(inp), *d, opts=bqc.make_opts(f_ov=f_dev), e_triplet=et)
    assert abs(e - e_ref) <= e_tol(e_ref)
    n = len(trip_ref)
    assert np.all(np.abs(et.cpu().numpy() - trip_ref) <= 1e-10 * np.abs(trip_ref) + 1e-12 * abs(e_ref) / n + 1e-300)
    # without f_ov the canonical value comes back; the host entry point copies f_ov itself
    assert abs(bqc.bqc_t_energy_ex(*dims(inp), *d) - e_canon) <= e_tol(e_canon)
    host = [torch.from_numpy(np.ascontiguousarray(a)) for a in inp.arrays()]
    e_host, h2d, _ = bqc.bqc_t_energy_host(*dims(inp), *host, opts=bqc.make_opts(f_ov=torch.from_numpy(inp.f_ov)))
    assert e_host == e
    assert h2d == inp.nbytes() + inp.f_ov.nbytes
    # V element by element
    o = inp.nocc
    for (i, j, k) in [(0, 1, 2), (0, 0, o - 1), (2, 0, 1)]:
        W, V = bqc.bqc_t_debug_wv(*dims(inp), *d, i, j, k, f_ov=f_dev)
        Wr = orc.w_triplet(inp, i, j, k)
        _close(W, Wr)
        _close(V, orc.v_triplet(inp, i, j, k, Wr))
