"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/*.h declares;
host-only entry points (no compute calls) behave."""
import ctypes
import glob
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2502_17963_b200.build import build_library
    return build_library()


def _declared_symbols():
    names = set()
    for h in glob.glob(os.path.join(ROOT, "include", "*.h")):
        src = open(h).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(bqc_\w+)\s*\(", src))
    return sorted(names)


def test_header_declares_the_boundary():
    names = _declared_symbols()
    for must in ["bqc_t_energy", "bqc_t_energy_ex", "bqc_t_energy_host", "bqc_t_workspace_bytes",
                 "bqc_t_num_triplets", "bqc_t_triplet_index", "bqc_last_error", "bqc_error_string"]:
        assert must in names


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    for name in _declared_symbols():
        assert hasattr(L, name), f"{name} declared in include/ but not exported"


def test_no_torch_types_in_the_abi():
    src = open(os.path.join(ROOT, "include", "bqc_t.h")).read()
    assert "torch" not in src.lower().replace("pytorch tensors", "") or "at::" not in src
    assert "at::Tensor" not in src and "#include <torch" not in src


def test_triplet_indexing(libpath):
    import paper_2502_17963_b200 as bqc
    for o in (1, 2, 3, 6, 11):
        n = 0
        for i in range(o):
            for j in range(i, o):
                for k in range(j, o):
                    assert bqc.bqc_t_triplet_index(o, i, j, k) == n
                    n += 1
        assert bqc.bqc_t_num_triplets(o) == n == o * (o + 1) * (o + 2) // 6
    assert bqc.bqc_t_triplet_index(5, 2, 1, 3) == -1
    assert bqc.bqc_t_triplet_index(5, 0, 1, 5) == -1
    assert bqc.bqc_t_num_triplets(100) == 171700


def test_flop_model_matches_survey(libpath):
    import paper_2502_17963_b200 as bqc
    # F_W = [o(o+1)(o+2)/6 - o] 12 v^3 (v+o)
    for (o, v), fw in {(5, 19): 5.93e7, (20, 76): 7.69e11, (40, 152): 9.26e13, (80, 304): 1.146e16,
                       (100, 380): 5.424e16}.items():
        assert bqc.bqc_t_flops(o, v) == pytest.approx(fw, rel=2e-3)
        assert bqc.bqc_t_flops(o, v) == (o * (o + 1) * (o + 2) // 6 - o) * 12.0 * v ** 3 * (v + o)
    w = bqc.make_opts(occ_lo=2, occ_hi=6)
    assert bqc.bqc_t_flops(20, 76, w) == (4 * 5 * 6 // 6 - 4) * 12.0 * 76 ** 3 * 96


def test_sharding_partitions_triplets(libpath):
    import paper_2502_17963_b200 as bqc
    o = 7
    for nshard in (1, 2, 3, 8):
        seen = {}
        for i in range(o):
            for j in range(i, o):
                for k in range(j, o):
                    r = bqc.bqc_t_triplet_owner(o, nshard, i, j, k)
                    assert 0 <= r < nshard
                    seen[(i, j, k)] = r
        counts = [list(seen.values()).count(r) for r in range(nshard)]
        assert sum(counts) == bqc.bqc_t_num_triplets(o) and max(counts) - min(counts) <= 1
        total = sum(bqc.bqc_t_flops(o, 9, bqc.make_opts(shard_rank=r, shard_count=nshard)) for r in range(nshard))
        assert total == bqc.bqc_t_flops(o, 9)
    assert bqc.bqc_t_triplet_owner(o, 0, 0, 1, 2) == -1


def test_plan_and_workspace(libpath):
    import paper_2502_17963_b200 as bqc
    assert bqc.bqc_t_plan_occ_block(5, 19, 84) == 5
    bo5 = bqc.bqc_t_plan_occ_block(100, 380, 1680)
    # config 5: the (vv|ov) tensor (43.9 GB) is never resident: 4*Bo slabs only
    assert 1 <= bo5 <= 25
    ws5 = bqc.bqc_t_workspace_bytes(100, 380, 1680)
    assert 10e9 < ws5 < 150e9
    assert bqc.bqc_t_workspace_bytes(100, 380, 1680, bqc.make_opts(occ_block=2)) < ws5
    # invalid arguments are reported, not crashed on
    assert bqc.bqc_t_workspace_bytes(0, 19, 84) == 0 and bqc.bqc_last_error() == 1
    assert bqc.bqc_t_workspace_bytes(5, 19, 84, bqc.make_opts(occ_lo=3, occ_hi=2)) == 0
    assert bqc.bqc_last_error() == 9
    assert "option" in bqc.bqc_error_string(9)
    assert bqc.bqc_error_string(0) == "ok"


def test_w_builder_tiling_covers_every_extent_exactly_once(libpath):
    """split_n / split_m: segments are disjoint, ordered, cover [0, v) and pad as little as
    the tile shapes allow: N to the next multiple of 8 (>= 32), M rows to v (main) + a strip < one tile."""
    import paper_2502_17963_b200 as bqc
    for v in list(range(1, 420)) + [512, 777, 1320]:
        cols, rows = bqc.bqc_debug_tiling(v)
        assert 1 <= len(cols) <= 2 and 1 <= len(rows) <= 2
        # columns: contiguous segments of tiles 8*NF wide, NF in [4, 16]
        n = 0
        for (n0, ntiles, nf) in cols:
            assert n0 == n and ntiles >= 1 and 4 <= nf <= 16
            n += ntiles * 8 * nf
        assert n >= v and n == max(32, (v + 7) // 8 * 8)
        assert sum(c[1] for c in cols) == max(1, -(-((v + 7) // 8) // 16))       # fewest tiles
        # rows: contiguous m1 ranges, tp * tq = 128, tq >= 8
        m = 0
        for (m1_0, tiles_m1, tp, tq) in rows:
            assert m1_0 == m and tiles_m1 >= 1 and tp * tq == 128 and tq >= 8
            m += tiles_m1 * tp
        assert m >= v
        if len(rows) == 2:
            assert rows[0][1] * rows[0][2] == rows[1][0] < v          # main part is all full tiles
        padded = sum(t * tp * (-(-v // tq) * tq) for (_, t, tp, tq) in rows)
        single = min(-(-v // (128 // tq)) * (128 // tq) * (-(-v // tq) * tq) for tq in (8, 16, 32, 64, 128))
        assert padded <= single                                        # never worse than one tile shape


def test_block_triple_sharding_flop_model_partitions_the_work(libpath):
    import paper_2502_17963_b200 as bqc
    F = bqc.BQC_T_FLAG_SHARD_BLOCKS
    for (o, v, bo) in [(20, 76, 0), (100, 380, 0), (100, 380, 5), (7, 11, 2)]:
        total = bqc.bqc_t_flops(o, v)
        for world in (1, 2, 8):
            parts = [bqc.bqc_t_flops(o, v, bqc.make_opts(shard_rank=r, shard_count=world, occ_block=bo, flags=F))
                     for r in range(world)]
            assert sum(parts) == total
    # config 5, 8 shards: within a few per cent of an even split
    parts = [bqc.bqc_t_flops(100, 380, bqc.make_opts(shard_rank=r, shard_count=8, flags=F)) for r in range(8)]
    assert max(parts) / (sum(parts) / 8) < 1.05


def test_bench_traffic_table_is_keyed_by_the_source_hash(tmp_path, monkeypatch):
    """bench.py reports roofline.traffic only from a committed ncu capture of the sources the build came from
    (profiles/r2_traffic.csv); anything else is None with a reason — never a typed-in constant."""
    import hashlib
    import bench
    csrc = os.path.join(ROOT, "paper_2502_17963_b200", "csrc")
    h = hashlib.sha256()
    for f in sorted(os.listdir(csrc)):
        with open(os.path.join(csrc, f), "rb") as fh:
            h.update(fh.read())
    sha = h.hexdigest()[:12]
    prof = tmp_path / "profiles"
    prof.mkdir()
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    # no table
    val, why = bench.ncu_traffic(5, "ijk")
    assert val is None and "absent" in why
    # table of another build
    os.symlink(os.path.join(ROOT, "paper_2502_17963_b200"), tmp_path / "paper_2502_17963_b200")
    (prof / "r2_traffic.csv").write_text("config,schedule,kernel,src_sha,dram_read_bytes,dram_write_bytes,capture\n"
                                         "5,ijk,w_builder,000000000000,1,2,x.txt\n")
    val, why = bench.ncu_traffic(5, "ijk")
    assert val is None and "000000000000" in why
    # table of this build
    (prof / "r2_traffic.csv").write_text("config,schedule,kernel,src_sha,dram_read_bytes,dram_write_bytes,capture\n"
                                         f"5,ijk,w_builder,{sha},10,5,x.txt\n")
    val, why = bench.ncu_traffic(5, "ijk")
    assert val == 15.0 and sha in why
    assert bench.ncu_traffic(3, "ijk")[0] is None and bench.ncu_traffic(5, "abc")[0] is None


def test_no_alloc_sum_limit_is_enforced_before_any_device_work(libpath):
    """bqc_sum_fixed_noalloc (the allocation-free entry point): the size limit of its static scratch array is a
    host-side check, so it is reported without a GPU."""
    L = ctypes.CDLL(libpath)
    L.bqc_sum_fixed_noalloc_max.restype = ctypes.c_size_t
    L.bqc_sum_fixed_noalloc.restype = ctypes.c_int
    L.bqc_sum_fixed_noalloc.argtypes = [ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p, ctypes.c_void_p]
    L.bqc_error_detail.restype = ctypes.c_char_p
    nmax = L.bqc_sum_fixed_noalloc_max()
    assert nmax == 4096 * 4096
    assert L.bqc_sum_fixed_noalloc(None, nmax + 1, None, None) == 1          # BQC_ERR_INVALID_SIZE
    assert b"exceeds the maximum" in L.bqc_error_detail()
