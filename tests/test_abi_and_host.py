"""CPU-side checks (-m "not gpu"): the C-ABI library builds, loads and exports every symbol that
include/me.h declares; the header is plain C; the generator's exact colour algebra and diagram counts
agree with the oracle's independent numeric ones; host logic (layout transforms, sharding) incl. a
world_size-2 gloo run.  No compute call is made here (no GPU)."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="session")
def melib():
    import __graft_entry__
    __graft_entry__.build()
    import paper_2303_18244_b200 as me
    return me


def declared_functions():
    text = open(os.path.join(ROOT, "include", "me.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(me_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for required in ("me_create", "me_filter_helicities", "me_compute", "me_rambo", "me_philox_uniform", "me_destroy"):
        assert required in names


def test_library_exports_every_declared_symbol(melib):
    lib = ctypes.CDLL(melib.LIB_PATH)
    for name in declared_functions():
        assert hasattr(lib, name), "libme_b200.so does not export %s" % name
    assert set(melib.EXPORTS) == set(declared_functions())


def test_header_is_plain_c_and_struct_layout_matches_binding(melib, tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "me.h"\n#include <stdio.h>\n#include <stddef.h>\n'
                   'int main(void){printf("%zu %zu %zu %zu\\n", sizeof(me_info), sizeof(me_sm_params), offsetof(me_info, mass), offsetof(me_info, flops_per_helicity));return 0;}\n')
    exe = tmp_path / "t"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()
    assert int(out[0]) == ctypes.sizeof(melib.me_info)
    assert int(out[1]) == ctypes.sizeof(melib.me_sm_params)
    assert int(out[2]) == melib.me_info.mass.offset
    assert int(out[3]) == melib.me_info.flops_per_helicity.offset


def test_strerror_without_gpu(melib):
    L = melib.lib()
    assert L.me_strerror(0) == b"ok"
    assert b"filter" in L.me_strerror(melib.ME_ENOTFILTERED)


def test_null_arguments_are_rejected_without_touching_cuda(melib):
    L = melib.lib()
    assert L.me_create(1, None, None) == melib.ME_EINVAL
    assert L.me_destroy(None) == melib.ME_EINVAL
    assert L.me_get_info(None, None) == melib.ME_EINVAL
    assert L.me_compute(None, None, 0, 0, None, None) == melib.ME_EINVAL
    prm = melib.me_sm_params(**melib.DEFAULT_SM)
    h = ctypes.c_void_p(0)
    assert L.me_create(17, ctypes.byref(prm), ctypes.byref(h)) == melib.ME_EPROCESS


def test_binding_fails_loudly_without_cuda(melib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(RuntimeError):
        melib.MEContext(melib.ME_GG_TTX)


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2303_18244_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "liboracle" not in text, f


# ------------------------------------------------------------------ generator vs oracle (independent colour algebra)
@pytest.mark.parametrize("n,process,ndiag", [(2, 1, 3), (3, 2, 16), (4, 3, 123), (5, 4, 1240)])
def test_generator_topology_against_oracle(orc, n, process, ndiag):
    from paper_2303_18244_b200.codegen.topology import Topology
    T = Topology(n)
    assert T.ndiagrams == ndiag
    info = orc.info(process)
    assert T.ncol == info["ncol"] and len(T.Cl) == info["n_closures"]
    # exact Fierz colour matrix (generator) == numeric Gell-Mann colour matrix (oracle)
    C_gen = np.array(T.color_num, dtype=float) / T.color_denom
    C_orc = orc.color_matrix(process)
    assert np.abs(C_gen - C_orc).max() < 1e-10
    assert T.color_denom == {2: 3, 3: 9, 4: 54, 5: 324}[n]
    # every jamp coefficient is a unit Gaussian integer
    for c in T.Cl:
        for _, coef in c.jamp:
            assert coef in (1, -1, 1j, -1j)


def test_generated_flop_counts_are_recorded(melib):
    import json
    s = json.load(open(os.path.join(ROOT, "paper_2303_18244_b200", "csrc", "generated", "gen_summary.json")))
    assert s["gg_ttxgg"]["ndiagrams"] == 123 and s["gg_ttxggg"]["ndiagrams"] == 1240
    # SURVEY §8(d) estimated 27-42 k + colour for the plain recursion; the two-sided scheme needs ~20 k
    assert 1.5e4 < s["gg_ttxgg"]["flops_per_helicity"] < 6e4


def test_flops_tables_match_the_device_routines(tmp_path):
    """the generator's per-routine flop tables (codegen/emit.py FLOPS, emit_orbit.py FL, emit_orbit5.py FL5) are not free
    parameters: tests/flopcount/count_flops.cpp instantiates the routines of csrc/hel_amp.cuh on the host with a scalar type
    that counts every +, -, *, / it executes (SURVEY.md section 8(d) rule), and every table entry must equal that count"""
    from paper_2303_18244_b200.codegen import emit, emit_orbit, emit_orbit5
    exe = tmp_path / "count_flops"
    subprocess.run(["g++", "-std=c++17", "-O0", "-I", os.path.join(ROOT, "tests", "flopcount"), "-I", os.path.join(ROOT, "paper_2303_18244_b200", "csrc"),
                    os.path.join(ROOT, "tests", "flopcount", "count_flops.cpp"), "-o", str(exe)], check=True)
    counted = {}
    for line in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.splitlines():
        name, v = line.split()
        counted[name] = int(v)
    assert counted["spinor_ubar_plus"] == counted["spinor_ubar_minus"] == counted["spinor_v_plus"] == counted["spinor_v_minus"]
    assert counted["v4_current"] == counted["v4_current_1"] == counted["v4_current_2"]
    alias = dict(quark_step="quark_step2", spinor="spinor_ubar_plus")
    for table in (emit.FLOPS, emit_orbit.FL, emit_orbit5.FL5):
        for key, val in table.items():
            if key == "jamp_entry":          # one complex add into an accumulator
                assert val == 2
                continue
            assert val == counted[alias.get(key, key)], (key, val, counted[alias.get(key, key)])
    # literals the emitters use next to the tables: momentum sums (4 per padd / psub) and the per-event bases
    assert counted["padd"] == counted["psub"] == 4 and counted["wadd"] == counted["wsub"] == 8
    assert counted["gluon_basis"] <= 22 and counted["spinor_basis"] <= 20      # `fixed` charges 22 per gluon basis, 40 for two spinor bases


def test_helicity_walk_of_the_sharing_kernel():
    """ME_OPT_SHARE_CURRENTS: the walk is a permutation of the 64 helicities in which consecutive steps differ in exactly one
    helicity, the quark helicities flip most often, particle 0 last (parity pairing keeps the first half); the re-evaluation
    counts that enter flops_per_event_shared follow from it"""
    from paper_2303_18244_b200.codegen import emit_orbit as eo
    walk = eo.gray_walk()
    assert sorted(walk) == list(range(64))
    flips = [a ^ b for a, b in zip(walk, walk[1:])]
    assert all(bin(f).count("1") == 1 for f in flips)
    count = {b: sum(1 for f in flips if f == 1 << b) for b in range(6)}
    assert count[eo.T_BIT] == 32 and count[eo.TB_BIT] == 16 and count[5] == 1          # t fastest, then t~; gluon 0 (bit 5) slowest
    assert all(not (h >> 5) & 1 for h in walk[:32])
    # a gluon pair is re-evaluated 1 + flips(a) + flips(b) times, a current of all four gluons 16 times
    assert eo.walk_count(eo.dep_mask([0, 1])) == 1 + count[5] + count[4]
    assert eo.walk_count(eo.dep_mask([0, 1, 2, 3])) == 16
    assert eo.walk_count(eo.dep_mask([2], t=True)) == 1 + 32 + count[eo.lam_bit(2)]
    src, info = eo.emit_orbit_process()
    assert 0.5 * 64 * info["flops_per_helicity"] < info["flops_shared_event"] < 0.7 * 64 * info["flops_per_helicity"]


# ------------------------------------------------------------------ host logic
def test_aosoa_roundtrip_and_padding():
    import inputs
    rng = np.random.default_rng(0)
    for n in (1, 31, 32, 33, 100):
        p = rng.normal(size=(n, 6, 4))
        flat = inputs.aos_to_aosoa(p, 32)
        assert flat.size == ((n + 31) // 32) * 6 * 4 * 32
        assert np.array_equal(inputs.aosoa_to_aos(flat, n, 6, 32), p)
        # element (event e, particle k, component c) sits at page e/32, lane e%32
        e, k, c = n - 1, 3, 2
        assert flat[(e // 32) * 6 * 4 * 32 + (k * 4 + c) * 32 + e % 32] == p[e, k, c]


def test_shard_ranges_cover_exactly_once():
    from paper_2303_18244_b200.shard import shard_range
    for n in (0, 1, 31, 32, 33, 1000, 524288, 65536 + 5):
        for world in (1, 2, 3, 8):
            seen = np.zeros(n, dtype=int)
            for r in range(world):
                f, c = shard_range(n, r, world)
                assert f % 32 == 0 or c == 0
                seen[f:f + c] += 1
            assert (seen == 1).all()


def _gloo_worker(rank, world, port, n, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import oracle
    from paper_2303_18244_b200.shard import shard_range
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    first, cnt = shard_range(n, rank, world)
    # each rank generates ITS events from the global event index (counter-based Philox) — no exchange
    p, w = oracle.events(oracle.GG_TTX, cnt, seed=1, first_event=first)
    me = oracle.me(oracle.GG_TTX, p, nthreads=1)
    # the only collective: one double per rank for the cross-section estimate
    s = torch.tensor([float((w * me).sum()), float(cnt)], dtype=torch.float64)
    dist.all_reduce(s)
    gathered = [None] * world
    dist.all_gather_object(gathered, (first, me))
    if rank == 0:
        q.put((s.tolist(), gathered))
    dist.destroy_process_group()


def test_two_rank_gloo_sharding_reproduces_single_rank(orc):
    import torch.multiprocessing as mp
    n, world, port = 200, 2, 29511 + os.getpid() % 500
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_gloo_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    (tot, cnt), gathered = q.get(timeout=120)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    p_all, w_all = orc.events(orc.GG_TTX, n, seed=1)
    me_all = orc.me(orc.GG_TTX, p_all, nthreads=1)
    me_sharded = np.concatenate([m for _, m in sorted(gathered, key=lambda t: t[0])])
    assert cnt == n
    assert np.array_equal(me_sharded, me_all)            # bit-identical: same events, same arithmetic
    assert abs(tot / float((w_all * me_all).sum()) - 1) < 1e-13


def test_orbit_emitters_cover_every_diagram_term():
    """the orbit-looped emitters enumerate shapes x relabellings on their own; their amplitude-term counts must equal the
    closure counts of the generic diagram enumeration (159 for 4 gluons, 1890 for 5), their colour-flow count n!"""
    from paper_2303_18244_b200.codegen import emit_orbit, emit_orbit5
    from paper_2303_18244_b200.codegen.topology import Topology
    _, info4 = emit_orbit.emit_orbit_process()
    assert info4["namp"] == len(Topology(4).Cl) == 159 and info4["ncol"] == 24
    assert sum(info4["shapes"].values()) == 6 + 4 + 4 + 4 + 6 + 12 + 3 + 6
    _, info5 = emit_orbit5.emit_orbit5_process()
    assert info5["namp"] == len(Topology(5).Cl) == 1890 and info5["ncol"] == 120
    # shared-memory budgets: one 128-thread CTA (FP64) per SM must fit 227 KB for cfg 4 and for every cfg 5 kernel
    assert info4["smem_slots"] * 8 * 128 <= 227 * 1024
    assert all(k["slots"] * 8 * emit_orbit5.BLOCK1 <= 227 * 1024 for k in info5["kernels"])
    assert sum(k["amplitudes"] for k in info5["kernels"]) == 1890
    # FP64 kernels with a tensor-memory scratchpad: the slots below tm_slot0 stay in shared memory, the rest take two 32-bit TMEM
    # columns each.  Two CTAs per SM need 2 x (dynamic + 16 B static + 1 KB reserved) <= 228 KB and 2 x tm_cols <= 512 columns.
    def two_ctas(slot0, nslots, cols):
        return 2 * (slot0 * 8 * 128 + 16 + 1024) <= 228 * 1024 and 2 * cols <= 512 and 2 * (nslots - slot0) <= cols
    assert two_ctas(info4["tm_slot0"], info4["smem_slots"], info4["tm_cols"])
    k0, k1, k2 = info5["kernels"]
    assert two_ctas(k0["tm_slot0"], k0["slots"], k0["tm_cols"]) and two_ctas(k1["tm_slot0"], k1["slots"], k1["tm_cols"])
    assert k2["tm_slot0"] is None                               # FP32 / fallback kernel: shared memory only
    v = k2["fp64_variant"]                                      # FP64 variant: 48 accumulators in TMEM, one CTA per SM
    assert v["tm_slot0"] * 8 * 128 + 16 <= 227 * 1024 and 2 * (v["slots"] - v["tm_slot0"]) <= v["tm_cols"] <= 512


def test_cfg5_flop_count_does_not_depend_on_the_kernel_split(monkeypatch):
    """the algorithmic flop count of g g -> t t~ g g g (every current once, symmetric colour form, no staging adds) is a
    property of the method: spreading the three-gluon sub-trees over 1, 2 or 3 kernels changes the executed count only"""
    from paper_2303_18244_b200.codegen import emit_orbit5
    seen = {}
    for parts in (1, 2, 3):
        monkeypatch.setattr(emit_orbit5, "K1_PARTS", parts)
        _, info = emit_orbit5.emit_orbit5_process()
        seen[parts] = (info["flops_per_helicity"], info["flops_executed_per_helicity"])
        assert len(info["kernels"]) == parts + 2
    assert len({v[0] for v in seen.values()}) == 1
    assert seen[1][1] < seen[2][1] < seen[3][1]
    ncol = 120
    assert info["colour_flops"] == 2 * ncol * (ncol + 1) + 4 * ncol
    assert 1.0e5 < seen[1][0] < seen[1][1] < 2.5e5
