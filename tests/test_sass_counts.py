"""CPU test: the FP64 instruction counts behind the roofline line (sg_kernel_model: kFp64InstrPerPair, kFlopsPerPair,
kLinFp64InstrPerPair, kLinFlopsPerPair in csrc/) are recounted from `cuobjdump -sass` of the built library, so that a
kernel change cannot silently leave the roofline arithmetic stale.

Method: in the SASS of interaction_kernel<4> / interaction_lin_kernel<4> find the loops (backward branches).  The pair
loop is the innermost loop that holds MUFU.RSQ64H (one per (target, vertex) pair: the square-root seed); the chunk loop
is the smallest loop enclosing it.  FP64-pipe instructions = DFMA + DADD + DMUL (+ DSETP etc. if present);
FLOPs = 2 DFMA + DADD + DMUL.  Per pair = pair-loop count / pairs per trip; per (target, chunk) = (chunk loop - pair
loop trips) shared by kChunk = 16 pairs.
"""
import re
import shutil
import subprocess

import pytest

from paper_2001_02765_b200 import binding

K_CHUNK = 16          # vertices per chunk (csrc/sg_layout.h kChunk), restated
T = 4                 # targets per thread of the <4> instantiations


def _sass(kernel_substr):
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    out = subprocess.run([exe, "-sass", binding.lib_path()], capture_output=True, text=True, check=True).stdout
    blocks = re.split(r"\n\s*Function : ", out)
    hit = [b for b in blocks if b.split("\n", 1)[0].find(kernel_substr) >= 0]
    assert len(hit) == 1, (kernel_substr, [b.split("\n", 1)[0] for b in hit])
    ins = []
    for m in re.finditer(r"/\*([0-9a-f]{4,})\*/\s+(.*?);", hit[0]):
        ins.append((int(m.group(1), 16), m.group(2).strip()))
    return ins


def _loops(ins):
    """(start, end) address ranges of backward branches."""
    out = []
    for addr, text in ins:
        m = re.search(r"\bBRA(?:\.\S+)?\s+(?:\S+,\s*)?(0x[0-9a-f]+)", text)
        if m and int(m.group(1), 16) < addr:
            out.append((int(m.group(1), 16), addr))
    return out


def _count(ins, lo, hi):
    c = {"DFMA": 0, "DADD": 0, "DMUL": 0, "RSQ": 0, "OTHER_FP64": 0}
    for addr, text in ins:
        if lo <= addr <= hi:
            op = re.sub(r"^@!?U?P\d+\s+", "", text).split()[0]
            base = op.split(".")[0]
            if base in ("DFMA", "DADD", "DMUL"):
                c[base] += 1
            elif base in ("DSETP", "DMNMX", "D2I", "I2D", "D2F", "F2D") or base.startswith("DMMA"):
                c["OTHER_FP64"] += 1
            if op.startswith("MUFU.RSQ64H"):
                c["RSQ"] += 1
    return c


def _per_pair(kernel_substr):
    ins = _sass(kernel_substr)
    loops = _loops(ins)
    with_rsq = [(hi - lo, lo, hi) for lo, hi in loops if _count(ins, lo, hi)["RSQ"] > 0]
    assert with_rsq, "no loop with MUFU.RSQ64H found"
    with_rsq.sort()
    _, plo, phi = with_rsq[0]                                   # pair loop = smallest such loop
    pair = _count(ins, plo, phi)
    enclosing = [(hi - lo, lo, hi) for lo, hi in loops if lo <= plo and hi >= phi and (lo, hi) != (plo, phi)]
    enclosing.sort()
    _, clo, chi = enclosing[0]                                  # chunk loop
    chunk = _count(ins, clo, chi)
    n_pairs = pair["RSQ"]                                       # pairs per trip of the pair loop
    assert n_pairs % T == 0 and (K_CHUNK * T) % n_pairs == 0
    assert pair["OTHER_FP64"] == 0 and chunk["OTHER_FP64"] == 0
    trips = K_CHUNK * T // n_pairs
    per_pair = {k: pair[k] / n_pairs for k in ("DFMA", "DADD", "DMUL")}
    # straight-line code of the chunk loop outside the pair loop, per (target, chunk)
    per_chunk = {k: (chunk[k] - pair[k]) / T for k in ("DFMA", "DADD", "DMUL")}
    instr = sum(per_pair.values()) + sum(per_chunk.values()) / K_CHUNK
    flops = (2 * per_pair["DFMA"] + per_pair["DADD"] + per_pair["DMUL"]
             + (2 * per_chunk["DFMA"] + per_chunk["DADD"] + per_chunk["DMUL"]) / K_CHUNK)
    return per_pair, per_chunk, instr, flops, trips


@pytest.mark.parametrize("kernel,substr", [(0, "interaction_kernelILi4E"), (1, "interaction_lin_kernelILi4E")])
def test_fp64_instruction_counts_match_the_sass(kernel, substr):
    per_pair, per_chunk, instr, flops, _ = _per_pair(substr)
    model_instr, model_flops = binding.kernel_instruction_counts(kernel)
    assert abs(instr - model_instr) < 1e-9, (per_pair, per_chunk, instr, model_instr)
    assert abs(flops - model_flops) < 1e-9, (per_pair, per_chunk, flops, model_flops)


def test_direct_kernel_uses_tma_and_no_libdevice_calls():
    ins = _sass("interaction_kernelILi4E")
    ops = [re.sub(r"^@!?U?P\d+\s+", "", t).split()[0] for _, t in ins]
    assert any(o.startswith("UBLKCP") for o in ops)            # cp.async.bulk (TMA bulk copy) of the vertex tiles
    assert not any(o.startswith("CALL") for o in ops)          # sqrt / log are inlined (no libdevice slow paths)
