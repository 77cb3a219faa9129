"""The roofline numerator is counted in the SASS of the library that was just built
(paper_2602_20787_b200/sassmix.py -> libsteps_cyl.sassmix.json), not written into bench.py.  CPU only:
cuobjdump disassembles without a GPU."""
import itertools
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def mix():
    from paper_2602_20787_b200 import build, sassmix
    build.build()
    assert os.path.exists(build.SASSMIX), "build.py must write the tally beside the library"
    # the committed tally is that of THIS binary: re-counting gives the same numbers
    again = sassmix.tally(build.LIB)
    data = sassmix.load(build.SASSMIX)
    assert again["kernels"] == data["kernels"]
    assert data["library_sha256"] == sassmix.file_sha256(build.LIB) and sassmix.is_current(build.LIB, build.SASSMIX)
    return data


def every_selectable_kernel():
    """Every name steps_cyl_pair_kernel_name() can return (steps_cyl.cu: name_pair_kernel)."""
    names = []
    for nc in range(0, 9):
        names += ["pair_fp64_sym_kernel<%d,%s,%d,false>" % (nc, o2, tr) for o2 in ("false", "true") for tr in (1, 2)]
        names += ["pair_fp64_sym_kernel<%d,false,%d,true>" % (nc, tr) for tr in (1, 2)]
        names += ["pair_fp64_round_kernel<%d,%s>" % (nc, sp) for sp in ("false", "true")]
        names += ["pair_mixed_round_kernel<%d,%s>" % (nc, sp) for sp in ("false", "true")]
        names += ["pair_fp64_kernel<%d>" % nc, "pair_mixed_kernel<%d>" % nc, "pair_mixed_sym_kernel<%d>" % nc]
    for ip, sched in itertools.product((0, 1), ("sym", "round")):       # CIC and TSC
        names += ["pair_table_%s_kernel<%d,4,false>" % (sched, ip), "pair_table_%s_kernel<%d,16,true>" % (sched, ip),
                  "pair_table_mixed_%s_kernel<%d>" % (sched, ip)]
    return names


def test_tally_covers_every_kernel_bench_can_select(mix):
    from paper_2602_20787_b200 import sassmix
    for name in every_selectable_kernel():
        assert name in mix["kernels"], name
        cnt, how = sassmix.per_interaction(mix, name, 12 if "<0," in name or name.endswith("<0>") else 5)
        arith = cnt["fp64_instr"] + cnt["fp32_ops"]
        assert arith > 5 and cnt["mufu"] >= 1, (name, cnt)
        assert cnt["fp64_flops"] >= cnt["fp64_instr"] - cnt["fp64_instr"] / 4      # DSETP carry no flop


def test_default_fp64_kernel_count(mix):
    """pair_fp64_sym_kernel<5,false>: one ring step = 2 unordered pairs = 4 interactions; the design's count is
    108 FP64-pipe instructions per unordered pair; a regression in either direction shows."""
    k = mix["kernels"]["pair_fp64_sym_kernel<5,false,2,false>"]
    m = k["mainline"]
    assert m.get("SHFL", 0) % 6 == 0 and m["SHFL"] >= 6      # three double accumulators travel: 6 SHFL per ring step
    steps = m["SHFL"] // 6                                   # ring steps in one (possibly unrolled) loop iteration
    assert k["interactions_per_iteration"] == 4 * steps and not k["nested"]
    per_unordered = 2 * k["per_interaction"]["fp64_instr"]
    assert per_unordered <= 110, per_unordered
    assert m.get("MUFU.RSQ64H", 0) == 20 * steps          # 10 images x 2 targets per ring step
    # the spline slow path is behind its pre-test, outside the mainline
    assert sum(k["slowpath"].values()) > 0 and "CALL" in k["slowpath"]


def test_per_image_cost_from_unrolled_instances(mix):
    from paper_2602_20787_b200 import sassmix
    for fam, lo, hi in (("pair_fp64_sym_kernel<%d,false,2,false>", 8.0, 10.5), ("pair_fp64_kernel<%d>", 17.0, 21.0)):
        d = (mix["kernels"][fam % 8]["per_interaction"]["fp64_instr"]
             - mix["kernels"][fam % 7]["per_interaction"]["fp64_instr"])
        assert lo <= d <= hi, (fam, d)              # two more images per pair evaluation
    c20, how = sassmix.per_interaction(mix, "pair_fp64_sym_kernel<0,false,2,false>", 20)
    c8, _ = sassmix.per_interaction(mix, "pair_fp64_sym_kernel<8,false,2,false>", 8)
    assert "extrapolated" in how and c20["fp64_instr"] > 2.2 * c8["fp64_instr"]


def test_bench_has_no_hard_coded_tallies():
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert "KERNEL_MIX" not in src and "NCU_DRAM_BYTES" not in src
    assert not re.search(r"dfma\s*=\s*\d", src)
    assert "sassmix" in src and "ncu_dram_traffic.csv" in src
    # every traffic row names the capture it came from
    import csv
    with open(os.path.join(ROOT, "profiles", "ncu_dram_traffic.csv")) as f:
        rows = list(csv.DictReader(l for l in f if not l.startswith("#")))
    assert rows
    for r in rows:
        assert os.path.exists(os.path.join(ROOT, r["source"])), r
        assert float(r["dram_bytes_read"]) > 0
