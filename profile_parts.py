"""Per-part instruction table of dies_fly from an ncu source page, and the work-per-unit constants of bench.py.

    ncu -i prof.ncu-rep --page source --csv --print-source cuda,sass > source.csv
    python profile_parts.py source.csv --counts crossings scatterings absorptions packages

The kernel source is cut into parts at anchor comments of csrc/dies_fly.cuh (found by their text in the file, which
must be the profiled one, so the table does not depend on line numbers).  Every SASS instruction belongs to the part of the nearest preceding instruction (in
address order) that comes from a line of dies_fly.cuh: the inlined helpers of dies_tracker.cuh (Philox, free paths,
table searches) are thereby counted with the part that calls them.  "Work" per unit:
  crossing    SASS instructions of one crossing step on a live lane (listed with --sass)
  scattering  predicated-on thread-instructions of the scattering branch + its share of the code the two event types
              have in common, per scattering
  absorption  the same for the absorption branch
  package     predicated-on thread-instructions of the source routine (escape tally, id fetch, launch) per package
Stack handling, batch composition, slot load / store, block ends and idle lanes are not work.
This module only reads a text file; it needs neither CUDA nor the library."""
from __future__ import annotations

import argparse
import csv
import os
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
from paper_2408_13807_b200.build import CSRC as HERE, KERNEL_SOURCES, kernel_hash  # noqa: E402  (the hash guard lives with the build)

# (part, anchor text that starts it), in source order
ANCHORS = [
    ("ev_sched", "// EVENT phase: typed batches"),
    ("ev_load", "// ---- the package of the slot"),
    ("ev_common", "if (!issrc) {"),
    ("ev_abs", "// (1) add the package's quantum to the shell tally"),
    ("ev_common", "if (act) {\n"),                     # second anchor of this text: the event proper (see SUB below)
    ("ev_src", "escape tally (L87 last sentence) + launch"),
    ("ev_store", "// ---- the package goes back into its slot"),
    ("cross_pop", "// CROSSING phase (PAPER.md L67-71"),
    ("cross_step", "// ---- kSteps crossings."),
    ("cross_end", "lc8 += pa - pb;"),
    ("flush", "// counters: flush before a 32-bit count can wrap"),
]
# the second workload: dies_tmc (csrc/dies_tmc.cuh), chosen with --kernel tmc
TMC_ANCHORS = [
    ("launch", "// ---- idle lanes launch new packages together"),
    ("guard", "// L119: a package ends below 1e-10"),             # (a lambda, inlined after the step and the scattering)
    ("cross", "// ---- kTmcSteps crossings of every active lane"),
    ("scatter", "// ---- scattering (L85): new direction"),
    ("flush", "// ---- flush the block's privatised tallies"),
]
SRC = "dies_fly.cuh"          # file the parts are cut in (main() switches it for --kernel tmc)

# sub-ranges inside the common event code that belong to one event type only
SUB = [
    ("ev_abs", "int row;", "blk = b + 1u;", 2),          # rows of the table, extra Philox block, draw
    ("ev_sca", "// ---- scattering with the HG phase function", "record<TRACE>(tp, pkg, n_ev, isabs", 0),
]


def _num(x: str) -> float:
    try:
        return float(x)
    except ValueError:
        return 0.0


def read_source_page(path: str):
    """-> (source lines of dies_fly.cuh {line: text}, SASS rows [(addr, file, line, sass, inst, thread, pred_on, samples)])."""
    src, sass = {}, []
    f, ix, ln = None, None, 0
    for r in csv.reader(open(path, newline="")):
        if not r:
            continue
        if r[0] == "File Path":
            f = os.path.basename(r[1]); continue
        if r[0] == "Function Name":
            continue
        if r[0] == "Line No":
            ix = {h: i for i, h in enumerate(r)}; continue
        if ix is None or len(r) < 4:
            continue
        if r[0].strip().isdigit():                      # a source line; the SASS rows that belong to it follow
            ln = int(r[0])
            if f == SRC:
                src.setdefault(ln, r[1])
            continue
        if r[0] == "" and r[2].startswith("0x") and len(r) > ix["# Samples"]:
            sass.append((int(r[2], 16), f, ln, r[3].strip(), _num(r[ix["Instructions Executed"]]),
                         _num(r[ix["Thread Instructions Executed"]]),
                         _num(r[ix["Predicated-On Thread Instructions Executed"]]), _num(r[ix["# Samples"]])))
    # an instruction is listed under every source line of its inline stack: keep one row per address, the one of
    # dies_fly.cuh when there is one (the caller), so that nothing is counted twice
    best = {}
    for row in sass:
        cur = best.get(row[0])
        if cur is None or (row[1] == SRC and cur[1] != SRC):
            best[row[0]] = row
    return src, sorted(best.values())


def part_of_lines(src: dict) -> dict:
    """Line of dies_fly.cuh -> part, from the anchors."""
    lines = sorted(src)
    text = {ln: src[ln] for ln in lines}

    def find(anchor, after=0, nth=0):
        a = anchor.strip()
        hits = [ln for ln in lines if ln > after and a in text[ln]]
        if not hits:
            raise SystemExit(f"anchor not found in the profiled source: {anchor!r}")
        return hits[nth]

    starts, last = [], 0
    for part, anchor in ANCHORS:
        ln = find(anchor, last)
        starts.append((ln, part)); last = ln
    part = {}
    for ln in lines:
        p = None                     # lines before the first anchor (set-up; address arithmetic the compiler
        for s, name in starts:       # re-materialises inside the loops) take the part of the code around them
            if ln >= s:
                p = name
        part[ln] = p
    for name, a0, a1, back in SUB:
        l0 = find(a0) - back
        l1 = find(a1, l0)
        for ln in lines:
            if l0 <= ln < l1:
                part[ln] = name
    return part


def table(path: str):
    src, sass = read_source_page(path)
    # the page lists only the lines that own instructions: the anchors are looked up in the file itself, which must
    # be the profiled one
    disk = {i + 1: t.rstrip("\n") for i, t in enumerate(open(os.path.join(HERE, SRC)))}
    for ln, t in src.items():
        if not disk.get(ln, "").replace('"', "").strip().startswith(t.replace('"', "").strip()):   # (ncu drops the quotes)
            raise SystemExit(f"csrc/{SRC} differs from the profiled source at line {ln}: re-profile this commit")
    lp = part_of_lines(disk)
    agg, cur = {}, "setup"
    rows = []
    for addr, f, ln, text, inst, thr, on, smp in sass:
        if f == SRC and lp.get(ln):
            cur = lp[ln]
        a = agg.setdefault(cur, [0.0, 0.0, 0.0, 0.0, 0])
        a[0] += inst; a[1] += thr; a[2] += on; a[3] += smp; a[4] += 1
        rows.append((addr, cur, text, inst, thr, on))
    return agg, rows


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("source_csv")
    ap.add_argument("--counts", type=float, nargs=4, metavar=("CROSSINGS", "SCATTERINGS", "ABSORPTIONS", "PACKAGES"),
                    help="event counts of the profiled launch (dies_get_counters)")
    ap.add_argument("--sass", action="store_true", help="list the SASS of the crossing block with its executed counts")
    ap.add_argument("--kernel", default="fly", choices=["fly", "tmc"],
                    help="fly: dies_fly (default); tmc: dies_tmc, --counts CROSSINGS SCATTERINGS 0 PACKAGES")
    a = ap.parse_args(argv)
    if a.kernel == "tmc":
        return main_tmc(a)
    agg, rows = table(a.source_csv)
    tot = sum(v[0] for v in agg.values()); smp = sum(v[3] for v in agg.values())
    print(f"kernel sources sha256 {kernel_hash()}")
    print(f"total warp-instructions {tot:.6g}, samples {smp:.0f}")
    print("| part | SASS instr | warp-instr % | samples % | active lanes | predicated-on lanes | pred-on thread-instr |")
    print("|---|---|---|---|---|---|---|")
    order = ["setup", "ev_sched", "ev_load", "ev_common", "ev_abs", "ev_sca", "ev_src", "ev_store", "cross_pop",
             "cross_step", "cross_end", "flush"]
    for p in order:
        if p in agg:
            v = agg[p]
            print(f"| {p} | {v[4]} | {100 * v[0] / tot:.1f} | {100 * v[3] / max(smp, 1):.1f} | {v[1] / max(v[0], 1):.1f} | "
                  f"{v[2] / max(v[0], 1):.1f} | {v[2]:.4g} |")
    if a.counts:
        nc, ns, na, npk = a.counts
        common = agg.get("ev_common", [0] * 5)[2] / max(ns + na, 1)
        i_s = common + agg.get("ev_sca", [0] * 5)[2] / max(ns, 1)
        i_a = common + agg.get("ev_abs", [0] * 5)[2] / max(na, 1)
        i_p = agg.get("ev_src", [0] * 5)[2] / max(npk, 1)
        step = [r for r in rows if r[1] == "cross_step"]
        blocks = max(r[3] for r in step)
        i_c_exec = sum(r[5] for r in step) / nc
        work = sum(agg.get(p, [0] * 5)[2] for p in ("ev_common", "ev_abs", "ev_sca", "ev_src"))
        print(f"executed thread-instr per crossing in cross_step: {sum(r[4] for r in step) / nc:.2f} issued, {i_c_exec:.2f} "
              f"predicated on ({blocks:.4g} blocks of the step loop)")
        print(f"I_scattering = {i_s:.1f} (common {common:.1f})")
        print(f"I_absorption = {i_a:.1f}")
        print(f"I_package    = {i_p:.1f}")
        print(f"event work {work:.4g} pred-on thread-instr = {100 * work / (32 * tot):.1f} % of the issued lane slots")
    if a.sass:
        print("\ncrossing block (cross_step), address order: executed warp-instr, SASS")
        for addr, p, text, inst, thr, on in rows:
            if p == "cross_step":
                print(f"{addr & 0xfffff:6x} {inst:12.0f}  {text}")


def main_tmc(a):
    """dies_tmc: one lane follows one package, so the parts are simply launch / crossing step / scattering / guard."""
    import hashlib
    global SRC, ANCHORS, SUB
    SRC, ANCHORS, SUB = "dies_tmc.cuh", TMC_ANCHORS, []
    agg, rows = table(a.source_csv)
    tot = sum(v[0] for v in agg.values()); smp = sum(v[3] for v in agg.values())
    print(f"csrc/dies_tmc.cuh sha256 {hashlib.sha256(open(os.path.join(HERE, SRC), 'rb').read()).hexdigest()}")
    print(f"total warp-instructions {tot:.6g}, samples {smp:.0f}")
    print("| part | SASS instr | warp-instr % | samples % | active lanes | predicated-on lanes | pred-on thread-instr |")
    print("|---|---|---|---|---|---|---|")
    for p in ["setup", "launch", "cross", "scatter", "guard", "flush"]:
        if p in agg:
            v = agg[p]
            print(f"| {p} | {v[4]} | {100 * v[0] / tot:.1f} | {100 * v[3] / max(smp, 1):.1f} | {v[1] / max(v[0], 1):.1f} | "
                  f"{v[2] / max(v[0], 1):.1f} | {v[2]:.4g} |")
    if a.counts:
        nc, ns, _, npk = a.counts
        get = lambda k: agg.get(k, [0] * 5)[2]
        print(f"I_crossing   = {(get('cross') + get('guard')) / max(nc, 1):.1f}  (step + continuous absorption + guard, per crossing)")
        print(f"I_scattering = {get('scatter') / max(ns, 1):.1f}")
        print(f"I_package    = {get('launch') / max(npk, 1):.1f}")
        work = get('cross') + get('guard') + get('scatter') + get('launch')
        print(f"work {work:.4g} pred-on thread-instr = {100 * work / (32 * tot):.1f} % of the issued lane slots")


if __name__ == "__main__":
    main()
