"""Instruction counts of the step loops, read from the SASS of the built library (cuobjdump -sass).

    python -m paper_1802_05065_b200.sasscount [--write]

For every integrator kernel in libfpt_b200.so this finds the innermost loops (a backward branch with no other backward
branch inside its body), takes the one with the most floating-point instructions -- the unrolled step loop -- and counts
its instructions by class.  Divided by the steps one trip integrates (persistent kernel: 4 macro steps = 8 steps in fp64,
16 in fp32; specialised kernel: the consumer loop does 8 steps per trip, the producer loop 2 Philox blocks = 4 / 8 steps)
this gives the instructions per trajectory step that bench.py sets beside the reference counts of SURVEY.md 8(a):

    fp64     DFMA DMUL DADD DSETP (+ MUFU.RCP64H / RSQ64H seeds are counted under "mufu")
    fp32     FFMA FMUL FADD FSETP (+ the packed FFMA2 / FMUL2 / FADD2, counted twice)

`--write` stores the table as profiles/sass_counts.json (build() does this), so the roofline's "executed instructions per
step" is reproducible from a tracked artefact and changes with the kernel, not with a constant typed into bench.py.
"""
from __future__ import annotations

import json
import re
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
LIB = HERE / "libfpt_b200.so"
OUT = HERE.parent / "profiles" / "sass_counts.json"

FP64 = ("DFMA", "DMUL", "DADD", "DSETP")
FP32 = ("FFMA", "FMUL", "FADD", "FSETP", "FFMA2", "FMUL2", "FADD2")
_INSTR = re.compile(r"^\s*/\*([0-9a-f]{4,})\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)\s*(.*?);")
_FUNC = re.compile(r"^\s*Function : (\S+)")


def _cuobjdump() -> str:
    for cand in ("/usr/local/cuda/bin/cuobjdump", "cuobjdump"):
        try:
            return subprocess.run([cand, "-sass", str(LIB)], capture_output=True, text=True, check=True).stdout
        except (FileNotFoundError, subprocess.CalledProcessError):
            continue
    raise RuntimeError("cuobjdump not found")


def _demangle(names):
    try:
        out = subprocess.run(["c++filt"], input="\n".join(names), capture_output=True, text=True, check=True).stdout.split("\n")
        return dict(zip(names, out))
    except Exception:
        return {n: n for n in names}


def _loops(instrs):
    """innermost loops as (start index, end index) over the instruction list"""
    addr_to_i = {a: i for i, (a, _, _) in enumerate(instrs)}
    back = []
    for i, (a, op, args) in enumerate(instrs):
        if op.startswith("BRA"):
            m = re.search(r"0x([0-9a-f]+)", args)
            if m:
                t = int(m.group(1), 16)
                if t <= a and t in addr_to_i:
                    back.append((addr_to_i[t], i))
    inner = [(s, e) for (s, e) in back if not any((s2, e2) != (s, e) and s <= s2 and e2 <= e for (s2, e2) in back)]
    return inner


def _classify(body):
    c = dict(total=len(body), fp64=0, fp32=0, mufu=0, imad_wide=0, imad=0, lop3=0, iadd_lea_shf=0, sel_mov=0, lds_sts=0, i2f_f2i=0,
             other=0)
    for _, op, _ in body:
        base = op.split(".")[0]
        if base in FP64:
            c["fp64"] += 1
        elif base in FP32:
            c["fp32"] += 2 if base.endswith("2") else 1
        elif base == "MUFU":
            c["mufu"] += 1
        elif base == "IMAD" and ".WIDE" in op:
            c["imad_wide"] += 1
        elif base == "IMAD":
            c["imad"] += 1
        elif base in ("LOP3", "PLOP3"):
            c["lop3"] += 1
        elif base in ("IADD3", "IADD", "LEA", "SHF", "IABS", "ISETP", "VIADD", "UIADD3"):
            c["iadd_lea_shf"] += 1
        elif base in ("SEL", "MOV", "UMOV", "R2UR", "PRMT", "CS2R", "FSEL", "FMNMX"):
            c["sel_mov"] += 1
        elif base in ("LDS", "STS", "LDC", "ULDC", "LDCU"):
            c["lds_sts"] += 1
        elif base in ("I2F", "F2I", "I2FP", "F2F", "F2FP"):
            c["i2f_f2i"] += 1
        else:
            c["other"] += 1
    return c


def count() -> dict:
    text = _cuobjdump()
    funcs, cur = {}, None
    for line in text.splitlines():
        m = _FUNC.match(line)
        if m:
            cur = m.group(1)
            funcs[cur] = []
            continue
        m = _INSTR.match(line)
        if m and cur is not None:
            funcs[cur].append((int(m.group(1), 16), m.group(2), m.group(3)))
    names = _demangle(list(funcs))
    table = {}
    for mangled, instrs in funcs.items():
        name = names[mangled]
        m = re.search(r"fpt_(persistent|specialised)_kernel<fpt::State(64|32)(?:X)?<(\d), ?(\d), ?(true|false), ?(true|false)(?:, ?(true|false))? ?>(, ?true)?", name)
        if not m:
            continue
        kind, prec, model, scheme, amp, ramp, fast, sliced = m.groups()
        fp32 = prec == "32"
        macro = 4 if fp32 else 2
        loops = [(s, e, _classify(instrs[s:e + 1])) for (s, e) in _loops(instrs)]
        loops = [l for l in loops if l[2]["fp64"] + l[2]["fp32"] >= 8]
        loops.sort(key=lambda l: -(l[2]["fp64"] + l[2]["fp32"]))
        key = f"{kind}_f{prec}_{'ud' if model == '1' else 'od'}_{('em', 'heun', 'paper')[int(scheme)]}_{'sin' if amp == 'true' else 'nosin'}_{'ramp' if ramp == 'true' else 'const'}" + ("_hwsin" if fast == "true" else "") + ("_sliced" if sliced else "")
        entry = {"kernel": name.split("(")[0]}

        def per_step(c, steps):
            d = {k: round(v / steps, 2) for k, v in c.items()}
            d["steps_per_trip"] = steps
            return d

        if kind == "persistent" and loops:
            # the step loop has the most floating-point work (the tail helper's served loop comes next when the variant has
            # one); macro steps per trip = Philox blocks per trip = IMAD.WIDE / 19 (20 per block, one folded by ptxas)
            blocks = max(1, round(loops[0][2]["imad_wide"] / 19.0))
            entry["step_loop"] = per_step(loops[0][2], blocks * macro)
        elif kind == "specialised" and len(loops) >= 2:
            cons = max(loops[:3], key=lambda l: l[2]["lds_sts"] > 0 and l[2]["imad_wide"] == 0)
            prod = max(loops[:3], key=lambda l: l[2]["imad_wide"])
            entry["consumer_loop"] = per_step(cons[2], 8)
            entry["producer_loop"] = per_step(prod[2], 2 * macro)
        table[key] = entry
    return table


def write(table=None) -> Path:
    """profiles/sass_counts.json"""
    table = count() if table is None else table
    OUT.parent.mkdir(exist_ok=True)
    OUT.write_text(json.dumps({"command": "python -m paper_1802_05065_b200.sasscount --write  (cuobjdump -sass of libfpt_b200.so)",
                               "per_step": table}, indent=1, sort_keys=True) + "\n")
    return OUT


def main():
    t = count()
    if "--write" in sys.argv:
        write(t)
    for k in sorted(t):
        e = t[k]
        for loop in ("step_loop", "consumer_loop", "producer_loop"):
            if loop in e:
                c = e[loop]
                print(f"{k:48s} {loop:14s} total {c['total']:7.2f}  fp64 {c['fp64']:6.2f}  fp32 {c['fp32']:6.2f}  imad.wide {c['imad_wide']:5.2f}  "
                      f"lop3 {c['lop3']:5.2f}  int {c['iadd_lea_shf'] + c['imad']:5.2f}  mov/sel {c['sel_mov']:5.2f}  mufu {c['mufu']:4.2f}  other {c['other']:5.2f}")


if __name__ == "__main__":
    main()
