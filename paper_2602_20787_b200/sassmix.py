"""Instruction mix of the pair kernels' inner loops, counted in the SASS of the built library.

    python -m paper_2602_20787_b200.sassmix [libsteps_cyl.so]      # prints the table, writes the JSON

`build.py` runs this after every compile and writes `libsteps_cyl.sassmix.json` beside the library;
`bench.py` takes the roofline numerator (FP64 / FP32 pipe instructions and flops per pair interaction,
SURVEY 8(d): "to be replaced by the SASS count of the shipped kernel") from that file, so an edit to a
kernel changes the numerator with it.

Method.  `cuobjdump -sass` lists every kernel; in each pair kernel the loops are the backward branches
(`BRA` to a lower address).  The PAIR LOOP is the loop that reads a source from shared memory (`LDS`),
contains no smaller loop that does, and holds the most arithmetic: one iteration of it evaluates
`pairs_per_iteration` pair terms (symmetric kernels: two targets of a lane against one source, each
result applied to both particles = 4 ordered interactions, times the ring steps an unrolled iteration holds -- read
off its shuffle count; ordered kernels: 1).  Instructions inside the
loop that a forward conditional branch can skip AND that lead to a CALL (the noinline spline of Eq. 3 behind
its pre-test: the slow path) are tallied separately as `slowpath`; everything else is the mainline count.
Kernels with a run-time image loop (template N_cut = 0) are marked `nested`: per_interaction() extrapolates
their counts in N_cut from the unrolled instances <8> and <7>.
"""
from __future__ import annotations

import json
import os
import re
import subprocess
import sys
from collections import Counter

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libsteps_cyl.so")
OUT = os.path.join(HERE, "libsteps_cyl.sassmix.json")

FP64_OPS = ("DFMA", "DMUL", "DADD", "DSETP")
FP32_OPS = ("FFMA", "FMUL", "FADD", "FFMA2", "FMUL2", "FADD2")

# kernel family -> ordered pair interactions one iteration of its pair loop evaluates
INTERACTIONS = {
    "pair_fp64_sym_kernel": 4, "pair_fp64_round_kernel": 4, "pair_mixed_sym_kernel": 4,
    "pair_mixed_round_kernel": 4, "pair_table_sym_kernel": 4, "pair_table_round_kernel": 4,
    "pair_table_mixed_sym_kernel": 4, "pair_table_mixed_round_kernel": 4,
    "pair_fp64_kernel": 1, "pair_mixed_kernel": 1,
}

_INS = re.compile(r"^\s+/\*([0-9a-f]{4,})\*/\s+(.*?)\s*;")
_BRA = re.compile(r"\bBRA(?:\.[A-Z.]+)?\s+(?:[!A-Z0-9]+,\s*)*0x([0-9a-f]+)")


def _tool(name):
    for c in (os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", name), name):
        if os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c):
            return c
    return name


def _demangle(names):
    try:
        out = subprocess.run([_tool("cu++filt"), *names], check=True, capture_output=True, text=True).stdout
        res = [l.strip() for l in out.splitlines()]
        if len(res) == len(names):
            return res
    except Exception:
        pass
    return list(names)


def _short(demangled):
    """'void steps::pair_fp64_sym_kernel<5, false>(...)' -> 'pair_fp64_sym_kernel<5,false>'."""
    m = re.search(r"steps::(\w+)(<[^>]*>)?", demangled)
    if not m:
        return demangled
    targs = (m.group(2) or "").replace(" ", "").replace("(bool)1", "true").replace("(bool)0", "false")
    targs = re.sub(r"\(int\)", "", targs)
    return m.group(1) + targs


def parse_functions(sass_text):
    """{mangled name: [(addr, predicate or None, opcode text)]}."""
    funcs, cur = {}, None
    for line in sass_text.splitlines():
        if "Function :" in line:
            cur = line.split("Function :")[1].strip()
            funcs[cur] = []
            continue
        if cur is None:
            continue
        m = _INS.match(line)
        if not m:
            continue
        text = m.group(2).strip()
        pred = None
        if text.startswith("@"):
            pred, text = text.split(None, 1)
        funcs[cur].append((int(m.group(1), 16), pred, text))
    return funcs


def _base(op):
    return op.split()[0].split(".")[0]


def analyse(ins):
    """Pair loop of one kernel: (start, end, mainline Counter, slow-path Counter, nested) or None."""
    # out-of-line device functions (the noinline spline, the general-path bodies) are listed after the kernel's
    # own code, from the lowest CALL target on: the pair loop is looked for in the kernel's own code only
    calls = [int(m.group(1), 16) for _, _, t in ins if t.startswith("CALL") for m in [re.search(r"0x([0-9a-f]+)", t)] if m]
    if calls:
        ins = [i for i in ins if i[0] < min(calls)]
    loops = []
    for a, pred, t in ins:
        m = _BRA.search(t)
        if m and t.startswith("BRA"):
            tgt = int(m.group(1), 16)
            if tgt <= a:
                loops.append((tgt, a))
    if not loops:
        return None
    def body(lo, hi):
        return [(a, p, t) for a, p, t in ins if lo <= a <= hi]
    def has_lds(lo, hi):
        return any(t.startswith("LDS") for _, _, t in body(lo, hi))
    cands = []
    for lo, hi in loops:
        if not has_lds(lo, hi):
            continue
        inner = [(l2, h2) for l2, h2 in loops if (l2, h2) != (lo, hi) and lo <= l2 and h2 <= hi]
        if any(has_lds(l2, h2) for l2, h2 in inner):
            continue
        b = body(lo, hi)
        arith = sum(1 for _, _, t in b if _base(t) in FP64_OPS + FP32_OPS or t.startswith("MUFU"))
        cands.append((arith, lo, hi, bool(inner)))
    if not cands:
        return None

    def tally_loop(lo, hi):
        b = body(lo, hi)
        # blocks a forward conditional branch inside the loop can skip; one that ends in a CALL (the noinline
        # spline of Eq. 3 behind its pre-test) is the slow path and is tallied apart, any other (e.g. the table
        # gathers only lanes inside rho_max take) counts as executed
        skip = []
        for a, pred, t in b:
            m = _BRA.search(t)
            if m and t.startswith("BRA") and pred is not None:
                tgt = int(m.group(1), 16)
                if a < tgt <= hi:
                    skip.append((a, tgt, any(t2.startswith("CALL") for a2, _, t2 in b if a < a2 < tgt)))
        main, skipped = Counter(), Counter()
        for a, pred, t in b:
            op = t.split()[0]
            key = _base(t)
            slow = any(s < a < e and call for s, e, call in skip)
            if key in ("DFMA", "DMUL", "DADD") and not slow:
                # distinct 64-bit REGISTER sources (not RZ / uniform registers / constants / immediates): an FP64
                # instruction with three of them issues over three cycles instead of two (measured)
                srcs = set(re.findall(r"(?<![U\w])R(\d+)", t.split(",", 1)[1] if "," in t else ""))
                if len(srcs) >= 3:
                    main["fp64_three_reg_sources"] += 1
                elif len(srcs) == 2:
                    main["fp64_two_reg_sources"] += 1
            if key == "MUFU":
                key = op                      # MUFU.RSQ / MUFU.RSQ64H / MUFU.RCP ...
            (skipped if slow else main)[key] += 1
        return main, skipped

    _, lo, hi, nested = max(cands)
    main, skipped = tally_loop(lo, hi)
    # variants of the pair loop: other candidate loops with the same rsqrt and shuffle counts (same pairs per
    # iteration), e.g. the SIMPLE ring pass of the mixed kernel; heaviest first, the main loop included
    def sig(c):
        return (sum(v for k, v in c.items() if k.startswith("MUFU")), c.get("SHFL", 0))
    variants = []
    for arith, l2, h2, _ in sorted(cands, reverse=True):
        m2, _s2 = tally_loop(l2, h2)
        if sig(m2) == sig(main):
            variants.append((l2, h2, m2))
    return lo, hi, main, skipped, nested, variants


def derive(kind_counts):
    c = kind_counts
    fp64_instr = sum(c.get(k, 0) for k in FP64_OPS)
    fp64_flops = 2 * c.get("DFMA", 0) + c.get("DMUL", 0) + c.get("DADD", 0)
    fp32_ops = 2 * (c.get("FFMA2", 0) + c.get("FMUL2", 0) + c.get("FADD2", 0)) \
        + c.get("FFMA", 0) + c.get("FMUL", 0) + c.get("FADD", 0)
    fp32_flops = 2 * (2 * c.get("FFMA2", 0) + c.get("FFMA", 0)) + 2 * (c.get("FMUL2", 0) + c.get("FADD2", 0)) \
        + c.get("FMUL", 0) + c.get("FADD", 0)
    fp32_issue = sum(c.get(k, 0) for k in FP32_OPS)
    mufu = sum(v for k, v in c.items() if k.startswith("MUFU"))
    conv = sum(v for k, v in c.items() if k in ("F2F", "F2I", "I2F", "F2FP"))
    three, two = c.get("fp64_three_reg_sources", 0), c.get("fp64_two_reg_sources", 0)
    # issue cycles of the FP64 instructions alone, with the measured costs per operand form (ubench_fp64_pipe.cu:
    # 2.0 cycles with at most one register source, 2.1 with two, 3.0 with three distinct ones)
    return dict(fp64_three_reg=three, fp64_two_reg=two, fp64_issue_cycles=2.0 * fp64_instr + 0.1 * two + 1.0 * three, fp64_instr=fp64_instr, fp64_flops=fp64_flops, fp32_ops=fp32_ops, fp32_flops=fp32_flops,
                fp32_issue=fp32_issue, mufu=mufu, conv=conv, total=sum(v for k, v in c.items() if not k.startswith("fp64_t")))


def file_sha256(path):
    import hashlib
    h = hashlib.sha256()
    with open(path, "rb") as f:
        for chunk in iter(lambda: f.read(1 << 20), b""):
            h.update(chunk)
    return h.hexdigest()


def is_current(lib_path=LIB, out_path=None):
    """True if the tally file beside `lib_path` was taken from exactly this binary."""
    out_path = out_path or os.path.splitext(lib_path)[0] + ".sassmix.json"
    try:
        return load(out_path).get("library_sha256") == file_sha256(lib_path)
    except (OSError, ValueError):
        return False


def tally(lib_path=LIB):
    sass = subprocess.run([_tool("cuobjdump"), "-sass", lib_path], check=True, capture_output=True,
                          text=True).stdout
    funcs = parse_functions(sass)
    names = list(funcs)
    kernels = {}
    for mangled, dem in zip(names, _demangle(names)):
        short = _short(dem)
        fam = short.split("<")[0]
        if fam not in INTERACTIONS:
            continue
        res = analyse(funcs[mangled])
        if res is None:
            continue
        lo, hi, main, skipped, nested, variants = res
        inter = INTERACTIONS[fam]
        if fam == "pair_fp64_sym_kernel":        # <N_cut, FAR_ORDER2, target tiles per CTA>: 2 interactions per target
            inter = 2 * int(short.rstrip(">").split(",")[2])
        if fam in ("pair_fp64_sym_kernel", "pair_fp64_round_kernel"):
            # the ring loop may be unrolled (STEPS_SYM_UNROLL): one ring step moves the source's three double
            # accumulators one lane down = 6 SHFL, so the shuffle count says how many steps an iteration holds
            inter *= max(1, main.get("SHFL", 0) // 6)
        d = derive(main)
        kernels[short] = {
            "loop": ["0x%04x" % lo, "0x%04x" % hi], "interactions_per_iteration": inter, "nested": nested,
            "mainline": dict(sorted(main.items())), "slowpath": dict(sorted(skipped.items())),
            "per_interaction": {k: v / inter for k, v in d.items()},
            # loops with the same pairs per iteration, heaviest first ([0] is the main loop)
            "variants": [{"loop": ["0x%04x" % l2, "0x%04x" % h2],
                          "per_interaction": {k: v / inter for k, v in derive(m2).items()}} for l2, h2, m2 in variants],
        }
    return {"library": os.path.basename(lib_path), "library_sha256": file_sha256(lib_path), "tool": "cuobjdump -sass",
            "kernels": kernels}


def write(lib_path=LIB, out_path=None):
    out_path = out_path or os.path.splitext(lib_path)[0] + ".sassmix.json"
    data = tally(lib_path)
    tmp = out_path + ".tmp.%d" % os.getpid()
    with open(tmp, "w") as f:
        json.dump(data, f, indent=1, sort_keys=True)
        f.write("\n")
    os.replace(tmp, out_path)
    return out_path


def load(path=OUT):
    """The tally of the built library (raises if build.py has not produced it)."""
    with open(path) as f:
        return json.load(f)


def per_interaction(mix, kernel, n_cut):
    """(counts per ORDERED pair interaction, how) for `kernel` as steps_cyl_pair_kernel_name() spells it.
    Image-mode kernels with the run-time image loop (first template argument 0, used for N_cut > 8) have a
    nested loop whose trip count is N_cut: their counts are extrapolated linearly in N_cut from the unrolled
    instances <8, ...> and <7, ...> of the same family."""
    ks = mix["kernels"]
    e = ks[kernel]
    fam, targs = kernel.split("<", 1)
    args = targs.rstrip(">").split(",")
    if fam.startswith("pair_table") or args[0] != "0":
        return dict(e["per_interaction"]), "counted"
    k8 = ks["%s<%s>" % (fam, ",".join(["8"] + args[1:]))]["per_interaction"]
    k7 = ks["%s<%s>" % (fam, ",".join(["7"] + args[1:]))]["per_interaction"]
    return ({k: k8[k] + (n_cut - 8) * (k8[k] - k7[k]) for k in k8},
            "extrapolated in N_cut from the unrolled <8> and <7> instances")


if __name__ == "__main__":
    lib = sys.argv[1] if len(sys.argv) > 1 else LIB
    path = write(lib)
    data = load(path)
    print("%-46s %-15s %5s %5s %5s %5s %6s %6s %5s %6s" % ("kernel", "loop", "DFMA", "DMUL", "DADD", "DSETP",
                                                            "fp32op", "MUFU", "all", "skip"))
    for k, v in sorted(data["kernels"].items()):
        m, p = v["mainline"], v["per_interaction"]
        i = v["interactions_per_iteration"]
        print("%-46s %-15s %5.1f %5.1f %5.1f %5.1f %6.1f %6.1f %5.1f %6d%s" % (
            k, "-".join(v["loop"]), m.get("DFMA", 0) / i, m.get("DMUL", 0) / i, m.get("DADD", 0) / i,
            m.get("DSETP", 0) / i, p["fp32_ops"], p["mufu"], p["total"], sum(v["slowpath"].values()),
            "  nested" if v["nested"] else ""))
    print("(per ordered pair interaction; written to %s)" % path)
