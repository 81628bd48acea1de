"""Epilogue instruction ledger by term (PAPER.md:437-445 table, 558 eps_mix, 876, 890).

  python -m paper_2606_23698_b200.ledger REPORT.ncu-rep --n-out N [--launch I] [--md OUT.md] [--lines OUT.csv]
  python -m paper_2606_23698_b200.ledger REPORT.ncu-rep --summary   # key raw metrics of every launch in the report
  python -m paper_2606_23698_b200.ledger --static            # SASS opcode histogram of the built library

REPORT is one `ncu --set full --import-source on` capture of ONE stage-kernel launch (the recipe in
profiles/*.md); N is the number of output-equivalents that launch produced (2 x complex elements: one
reconstructed real scalar each, Eq. 12).  The tool reads the report with `ncu -i`, attributes every
executed thread instruction to a step of SURVEY.md 8(a) through the `// [ledger: <term>]` markers in the kernel
sources (a marker applies to the lines below it until the next marker of that file; inlined functions keep the
markers of the file they are defined in), and prints

  * thread instructions per output-equivalent by term, beside the paper's model figures;
  * eps_mix: the executed instruction mix by issue class (alu / fma / lsu / xu / control / uniform+async), from the
    SASS opcodes of the same capture (PAPER.md:558 lets eps_mix range over [0.57, 1]);
  * c_q^res: deconstruction thread instructions per element and modulus (3.0 - 6.3);
  * the issue ceiling these counts imply at 148 SM x 128 lanes x 1.965 GHz.

Nothing here runs on the GPU and no module under oracle/ is used.
"""
import argparse
import collections
import csv
import glob
import io
import os
import re
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
MARK = re.compile(r"//\s*\[ledger:\s*(.+?)\s*\]")
DEFAULT_TERM = "setup, tile decode, loop control"
OTHER_FILES_TERM = "helpers from CUDA headers (shuffles, min/max, address conversion)"

# the paper's model, thread instructions per output-equivalent unless noted
PAPER_TERMS = [("deconstruction residual, per element (12 moduli)", "36-76"), ("dp4a deconstruction bulk, per element", "2-4"),
               ("canonicalise", "24-36"), ("residue combines", "30"), ("biased deposits + normalise", "66-70"),
               ("two-sided lift", "25-35"), ("correctly rounded pack", "20-30"), ("total c_epi", "203-281")]

CLASSES = [
    ("fma (IMAD / IMAD.WIDE / IMAD.HI, FFMA)", re.compile(r"^(IMAD|FFMA|FMUL|FADD|HFMA2|IMUL|IDP)")),
    ("alu (IADD3, LOP3, SHF, PRMT, ISETP, SEL, LEA, VIADD, VIMNMX, MOV)", re.compile(r"^(IADD|IADD3|LOP3|LOP|SHF|SHL|SHR|PRMT|ISETP|SEL|LEA|VIADD|VIMNMX|VIADDMNMX|MOV|IABS|IMNMX|PLOP3|CS2R|S2R|NOP|P2R|R2P|BMSK|SGXT|FSETP|FSEL)")),
    ("xu (FLO / POPC / conversions / MUFU)", re.compile(r"^(FLO|POPC|BREV|MUFU|I2F|F2I|F2F|I2I|FRND)")),
    ("lsu (LDG, STG, LDS, STS, LDC, ATOMS, shuffles)", re.compile(r"^(LDG|STG|LDS|STS|LDC|LD|ST|ATOM|ATOMS|RED|SHFL|LDSM|MATCH|VOTE|REDUX|LDL|STL|CCTL|MEMBAR|FENCE|ERRBAR)")),
    ("control (BRA, BSSY/BSYNC, BAR, WARPSYNC, EXIT, CALL/RET, nanosleep)", re.compile(r"^(BRA|BSSY|BSYNC|BAR|WARPSYNC|EXIT|CALL|RET|BRX|JMP|YIELD|NANOSLEEP|BREAK|DEPBAR|BPT)")),
    ("uniform datapath + async units (U*, UTC*, LDTM/STTM, SYNCS, UBLKCP, ELECT, R2UR)", re.compile(r"^(U[A-Z0-9]|LDTM|STTM|SYNCS|ELECT|R2UR|ACQBULK|ARRIVES|UTC)")),
]


def term_map():
    """{basename: [(first_line, term), ...]} from the markers in csrc/"""
    out = {}
    for f in sorted(glob.glob(os.path.join(CSRC, "*"))):
        marks = []
        for i, line in enumerate(open(f, errors="replace"), 1):
            m = MARK.search(line)
            if m:
                marks.append((i, m.group(1)))
        out[os.path.basename(f)] = marks
    return out


def term_of(tmap, fname, line):
    if fname not in tmap:
        return OTHER_FILES_TERM
    t = DEFAULT_TERM
    for start, name in tmap[fname]:
        if line >= start:
            t = name
    return t


LAUNCH = 0  # which launch of a multi-launch report to read (--launch)


def _ncu(args):
    if args[:1] == ["-i"]:
        args = args[:2] + ["--launch-skip", str(LAUNCH), "--launch-count", "1"] + args[2:]
    r = subprocess.run(["ncu"] + args, capture_output=True, text=True)
    if r.returncode != 0:
        raise SystemExit("ncu failed: " + r.stderr[-2000:])
    return r.stdout


def read_lines(report):
    """[(file, line, thread_inst, pred_on_thread_inst)] per source line and [(opcode, thread_inst)] per SASS instruction.
    The source page lists an inlined instruction under EVERY frame of its inline stack (call site, wrapper, callee line):
    each SASS address is counted once, under the innermost frame -- taken to be the listing line with the smallest
    aggregate, the most specific one."""
    rows = list(csv.reader(io.StringIO(_ncu(["-i", report, "--page", "source", "--csv", "--print-source", "sass,cuda"]))))
    f = None
    cur = None
    agg = {}                                  # (file, line) -> aggregate thread inst of the listing line
    seen = collections.defaultdict(list)      # address -> [(file, line)]
    own = {}                                  # address -> (thread inst, pred-on thread inst)
    for r in rows:
        if not r:
            continue
        if r[0] == "File Path":
            f = os.path.basename(r[1])
        elif r[0] == "Line No" and len(r) > 8:
            h = r
            it, ip, il, ia = h.index("Thread Instructions Executed"), h.index("Predicated-On Thread Instructions Executed"), h.index("Line No"), h.index("Address")
        elif f and r[0] not in ("Function Name",) and len(r) > 8:
            if r[il].strip():
                try:
                    cur = (f, int(r[il]))
                    agg[cur] = agg.get(cur, 0) + int(r[it])
                except ValueError:
                    cur = None
            elif cur and r[ia].startswith("0x"):
                try:
                    own[r[ia]] = (int(r[it]), int(r[ip]))
                    seen[r[ia]].append(cur)
                except ValueError:
                    pass
    per = collections.OrderedDict()
    for addr, places in seen.items():
        key = min(places, key=lambda k: agg.get(k, 0))
        a, b = per.get(key, (0, 0))
        per[key] = (a + own[addr][0], b + own[addr][1])
    ops = collections.Counter()
    rows = list(csv.reader(io.StringIO(_ncu(["-i", report, "--page", "source", "--csv", "--print-source", "sass"]))))
    hdr = None
    for r in rows:
        if r and r[0] == "Address":
            hdr = r
            io_, ii = hdr.index("Source"), hdr.index("Thread Instructions Executed")
        elif hdr and len(r) == len(hdr) and r[0].startswith("0x"):
            t = r[io_].split()
            if t:
                op = t[1] if t[0].startswith("@") and len(t) > 1 else t[0]
                ops[op.rstrip(";")] += int(r[ii] or 0)
    return [(k[0], k[1], v[0], v[1]) for k, v in per.items()], ops


def classify(op):
    base = op.split(".")[0]
    for name, rx in CLASSES:
        if rx.match(base):
            return name
    return "other"


def raw_metrics(report):
    rows = list(csv.reader(io.StringIO(_ncu(["-i", report, "--page", "raw", "--csv"]))))
    return dict(zip(rows[0], rows[-1]))


def report(path, n_out, moduli=12):
    tmap = term_map()
    lines, ops = read_lines(path)
    per = collections.Counter()
    on = collections.Counter()
    for f, l, n, p in lines:
        t = term_of(tmap, f, l)
        per[t] += n
        on[t] += p
    tot, tot_on = sum(per.values()), sum(on.values())
    raw = raw_metrics(path)
    o = []
    o.append(f"kernel: {raw.get('Kernel Name', '?')}  grid {raw.get('Grid Size', '?')}  duration {raw.get('gpu__time_duration.sum', '?')} ms")
    o.append(f"n_out (output-equivalents of the launch) = {n_out:.0f}")
    o.append("")
    o.append("Per-line counts come from ncu's instrumented replay (REPORT must hold ONE launch): the arithmetic terms are exact, but the kernel "
             "runs slower under instrumentation, so its waiting roles spin longer and the two `sync` terms are inflated; the un-instrumented "
             "total is the last line (warp instructions x 32 / n_out, hardware counter), and total minus the arithmetic terms is the real polling.")
    o.append("")
    o.append("| term (SURVEY.md 8(a)) | thread inst / output-eq | predicated-on | share |")
    o.append("|---|---|---|---|")
    for k, n in per.most_common():
        o.append(f"| {k} | {n / n_out:.1f} | {on[k] / n_out:.1f} | {n / tot * 100:.1f} % |")
    o.append(f"| **total (source-attributed)** | **{tot / n_out:.1f}** | **{tot_on / n_out:.1f}** | 100 % |")
    o.append("")
    decon = sum(n for k, n in per.items() if k.startswith(("a3", "a2")))
    o.append(f"deconstruction (a2 + a3) = {decon / n_out:.1f} thread inst per element -> c_q^res = {decon / n_out / moduli:.2f} per element and modulus "
             f"(paper: 3.0 - 6.3 residual + 2-4/12 dp4a bulk, PAPER.md:190, 441)")
    o.append("")
    o.append("paper's model for comparison (PAPER.md:437-445): " + "; ".join(f"{k} {v}" for k, v in PAPER_TERMS))
    o.append("")
    cls = collections.Counter()
    for op, n in ops.items():
        cls[classify(op)] += n
    ctot = sum(cls.values()) or 1
    o.append("| issue class (eps_mix, PAPER.md:558) | thread inst / output-eq | share |")
    o.append("|---|---|---|")
    for k, n in cls.most_common():
        o.append(f"| {k} | {n / n_out:.1f} | {n / ctot * 100:.1f} % |")
    o.append("")
    top = ", ".join(f"{op} {n / ctot * 100:.1f}%" for op, n in ops.most_common(14))
    o.append("most executed opcodes: " + top)
    o.append("")
    for k in ("smsp__inst_executed.sum", "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__warps_active.avg.pct_of_peak_sustained_active",
              "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
              "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
              "dram__bytes_read.sum", "dram__bytes_write.sum", "launch__registers_per_thread"):
        if k in raw:
            o.append(f"{k} = {raw[k]}")
    try:
        winst = float(raw["smsp__inst_executed.sum"])
        o.append(f"warp instructions x 32 / n_out = {winst * 32 / n_out:.1f} thread inst per output-eq (predicated-off lanes included)")
        o.append(f"issue ceiling at 148 SM x 128 lanes x 1.965 GHz = 37.2 T thread-inst/s: {winst * 32 / 37.22e12 * 1e3:.3f} ms for this launch")
    except Exception:
        pass
    return "\n".join(o), lines


def static_histogram(so):
    txt = subprocess.run(["cuobjdump", "-sass", so], capture_output=True, text=True, check=True).stdout
    per, name = collections.OrderedDict(), None
    for line in txt.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            per[name] = collections.Counter()
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]*)", line)
        if m and name:
            per[name][m.group(1).split(".")[0]] += 1
    o = ["| function | instructions | UTCIMMA | UTCCP | LDTM | UBLKCP | SYNCS | IMAD | IADD3 | LOP3 | SHF | PRMT | LDG | STG | LDS | STS | fp64 opcodes |", "|" + "---|" * 17]
    for k, c in per.items():
        short = re.sub(r"^_ZN2oz\d*", "", k)[:44]
        fp64 = sum(n for op, n in c.items() if re.match(r"^D(ADD|MUL|FMA|SETP|MNMX|MMA)$", op))
        o.append(f"| {short} | {sum(c.values())} | " + " | ".join(str(c.get(x, 0)) for x in
                 ("UTCIMMA", "UTCCP", "LDTM", "UBLKCP", "SYNCS", "IMAD", "IADD3", "LOP3", "SHF", "PRMT", "LDG", "STG", "LDS", "STS")) + f" | {fp64} |")
    return "\n".join(o)


SUMMARY_KEYS = [
    "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "lts__t_sector_hit_rate.pct",
    "smsp__inst_executed.sum", "smsp__thread_inst_executed.sum", "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "sm__warps_active.avg.pct_of_peak_sustained_active", "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "launch__registers_per_thread", "sm__cycles_elapsed.avg"]
STALLS = ["long_scoreboard", "wait", "barrier", "not_selected", "math_pipe_throttle", "branch_resolving", "short_scoreboard",
          "dispatch_stall", "no_instruction", "mio_throttle", "lg_throttle", "sleeping"]


def summary(report):
    """key raw metrics of EVERY launch in the report, one column per launch (markdown)"""
    r = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True)
    if r.returncode != 0:
        raise SystemExit("ncu failed: " + r.stderr[-2000:])
    rows = list(csv.reader(io.StringIO(r.stdout)))
    hdr, units, launches = rows[0], rows[1], rows[2:]
    o = ["| metric | unit | " + " | ".join(f"launch {i}" for i in range(len(launches))) + " |", "|---|---|" + "---|" * len(launches)]
    o.append("| kernel | | " + " | ".join(re.sub(r"\(.*", "", l[hdr.index("Kernel Name")])[-40:] + " grid " + l[hdr.index("Grid Size")] for l in launches) + " |")
    for k in SUMMARY_KEYS:
        if k in hdr:
            i = hdr.index(k)
            o.append(f"| {k} | {units[i]} | " + " | ".join(l[i] for l in launches) + " |")
    for st in STALLS:
        k = f"smsp__average_warps_issue_stalled_{st}_per_issue_active.ratio"
        if k in hdr:
            i = hdr.index(k)
            o.append(f"| stall {st} (warps per issue) | | " + " | ".join(f"{float(l[i]):.2f}" for l in launches) + " |")
    return "\n".join(o)


def kernel_source_hash():
    """sha256 over the kernel sources (csrc/*, include/*.h): ties a stored ncu figure to the code it was measured on"""
    import hashlib
    h = hashlib.sha256()
    root = os.path.dirname(_HERE)
    for f in sorted(glob.glob(os.path.join(CSRC, "*")) + glob.glob(os.path.join(root, "include", "*.h"))):
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def constants(report, key, n_out, out_json, command):
    """profiles/ncu_constants.json entry `key` (e.g. "bf:1024") from a report that holds ALL stage launches of one transform:
    DRAM bytes per launch (mean), thread instructions per output-equivalent (32 x warp instructions summed over the launches / n_out)."""
    import json
    r = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True)
    if r.returncode != 0:
        raise SystemExit("ncu failed: " + r.stderr[-2000:])
    rows = list(csv.reader(io.StringIO(r.stdout)))
    hdr, units, launches = rows[0], rows[1], rows[2:]

    def col(name, scale_units):
        i = hdr.index(name)
        return [float(l[i]) * scale_units.get(units[i], 1.0) for l in launches]
    byte_units = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    dram = [a + b for a, b in zip(col("dram__bytes_read.sum", byte_units), col("dram__bytes_write.sum", byte_units))]
    tinst = 32.0 * sum(col("smsp__inst_executed.sum", {}))  # warp instructions x 32: issue-slot equivalents (predicated-off lanes included)
    ms = col("gpu__time_duration.sum", {"ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3})
    try:
        db = json.load(open(out_json))
    except Exception:
        db = {}
    if db.get("source_hash") != kernel_source_hash():
        db = {"source_hash": kernel_source_hash(), "entries": {}}
    db["note"] = ("ncu figures bench.py quotes (never measured inside the timed run); valid only for the kernel sources with this hash "
                  "(paper_2606_23698_b200.ledger.kernel_source_hash), otherwise bench.py prints null")
    db["entries"][key] = {"dram_bytes_per_launch": sum(dram) / len(dram), "dram_bytes_per_launch_each": dram,
                          "thread_inst_per_output_eq": tinst / n_out, "launches": len(launches), "ncu_ms_per_launch": ms,
                          "n_out": n_out, "command": command}
    json.dump(db, open(out_json, "w"), indent=1)
    return json.dumps(db["entries"][key], indent=1)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report", nargs="?")
    ap.add_argument("--n-out", type=float)
    ap.add_argument("--md", help="write the tables to this file as well")
    ap.add_argument("--lines", help="write the per-line counts (file, line, term, thread inst, predicated-on) as CSV")
    ap.add_argument("--launch", type=int, default=0, help="index of the launch to read in a report that holds several (default 0)")
    ap.add_argument("--summary", action="store_true", help="key raw metrics of every launch in the report (no --n-out needed)")
    ap.add_argument("--constants", help="write / update this JSON (profiles/ncu_constants.json) from a report holding every stage launch of one transform")
    ap.add_argument("--key", help="entry name for --constants: VARIANT:SIZE, e.g. bf:1024 or bf-unfused:1024")
    ap.add_argument("--command", default="", help="the ncu command that made the report (recorded with --constants)")
    ap.add_argument("--static", action="store_true", help="SASS opcode histogram of libozfft.so (no report needed)")
    a = ap.parse_args()
    global LAUNCH
    LAUNCH = a.launch
    if a.static:
        out = static_histogram(os.path.join(_HERE, "libozfft.so"))
    elif a.constants:
        if not (a.report and a.n_out and a.key):
            ap.error("REPORT, --n-out and --key are required with --constants")
        out = constants(a.report, a.key, a.n_out, a.constants, a.command)
    elif a.summary:
        if not a.report:
            ap.error("REPORT is required")
        out = summary(a.report)
    else:
        if not a.report or not a.n_out:
            ap.error("REPORT and --n-out are required")
        out, lines = report(a.report, a.n_out)
        if a.lines:
            tmap = term_map()
            with open(a.lines, "w", newline="") as fh:
                w = csv.writer(fh)
                w.writerow(["file", "line", "term", "thread_inst", "pred_on_thread_inst"])
                for f, l, n, p in sorted(lines, key=lambda x: -x[2]):
                    if n:
                        w.writerow([f, l, term_of(tmap, f, l), n, p])
    print(out)
    if a.md:
        open(a.md, "w").write(out + "\n")


if __name__ == "__main__":
    sys.exit(main())
