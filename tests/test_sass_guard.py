"""CPU-side checks on the machine code of the fused decode kernel (cuobjdump -sass on the built library).

The consumer warps of the fused kernel hand a ring stage back to the producer with an mbarrier arrive.  That
arrive must not issue before the stage's fragment loads have returned (ptxas places a plain arrive
right behind the ISSUE of the last LDS, and the producer's refill then overwrites fragments still being read).
`release_stage` makes the barrier address depend on the accumulators the fragments feed; this test checks that
the dependence is there in the SASS ptxas actually produced, for every consumer arrive of the kernel."""
import re
import shutil
import subprocess

import pytest

from paper_2502_02040_b200 import build as _build


def _fused_sass():
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    out = subprocess.run([exe, "-sass", _build.build()], capture_output=True, text=True, check=True).stdout
    lines, on = [], False
    for ln in out.splitlines():
        if "Function :" in ln:
            on = "m2r2_fused_decode_kernel" in ln
            continue
        if on:
            m = re.match(r"\s+/\*[0-9a-f]+\*/\s+(.*?);", ln)
            if m:
                lines.append(m.group(1).strip())
    return lines


def _regs(tok):
    return re.findall(r"\bR(\d+)\b", tok)


def _dest_and_sources(ins):
    """-> (set of destination registers, set of source registers) of one SASS instruction (predicates dropped)."""
    ins = re.sub(r"^@!?U?P\d+\s+", "", ins)
    op, _, rest = ins.partition(" ")
    ops = [o.strip() for o in rest.split(",")]
    if not ops or not ops[0]:
        return op, set(), set()
    d = _regs(ops[0])
    dest = set()
    if d and not ops[0].startswith("["):
        base = int(d[0])
        width = 4 if (op.startswith("HMMA") or ".128" in op) else (2 if ".64" in op else 1)
        dest = {base + i for i in range(width)}
        srcs = set(int(r) for o in ops[1:] for r in _regs(o))
    else:
        srcs = set(int(r) for o in ops for r in _regs(o))
    return op, dest, srcs


def test_consumer_arrive_depends_on_the_stage_accumulators():
    sass = _fused_sass()
    assert sass, "m2r2_fused_decode_kernel not found in the library's SASS"
    arrives = [i for i, ins in enumerate(sass) if "SYNCS.ARRIVE.TRANS64.A1T0" in ins]
    assert len(arrives) >= 2, "expected the consumer arrives of the row-owned and the split-K GEMV loops"
    for i in arrives:
        addr = set(int(r) for r in _regs(sass[i].split("[")[1].split("]")[0]))
        # follow the address register's definitions upwards; the chain must reach an HMMA result
        need, found, depth = set(addr), False, 0
        j = i - 1
        while j >= 0 and need and depth < 400 and not found:
            op, dest, srcs = _dest_and_sources(sass[j])
            if dest & need:
                if op.startswith("HMMA"):
                    found = True
                    break
                if op.startswith(("LDS", "LDG", "LDC", "S2R", "MOV", "IMAD.MOV", "CS2R", "LEA", "SHF")) and not srcs:
                    need -= dest
                else:
                    need = (need - dest) | srcs
            j -= 1
            depth += 1
        assert found, "consumer arrive at SASS line %d does not depend on an HMMA result:\n%s" % (i, "\n".join(sass[max(0, i - 12):i + 1]))
        # and no fragment load of the ring between that HMMA and the arrive
        assert not any(x.startswith("LDS.128") for x in sass[j + 1:i]), "LDS.128 between the last dependent HMMA and the arrive"


def test_fused_kernel_uses_bulk_copies_and_tensor_pipe():
    """The instruction mix the design claims: bulk async copies (UBLKCP), mma.sync (HMMA), reds."""
    sass = _fused_sass()
    ops = " ".join(s.split(" ")[0] for s in sass)
    for mnemonic in ("UBLKCP", "HMMA.16816.F32.BF16", "REDG.E.ADD.F32", "LDGSTS"):
        assert mnemonic in ops or any(mnemonic in s for s in sass), mnemonic
