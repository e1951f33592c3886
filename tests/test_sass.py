"""Checks on the machine code nvcc produced for libspegg.so (-m "not gpu": cuobjdump runs without a GPU).

The C3 step draws its chunks from ONE global ticket: lane 0 of a warp takes it and the warp reads it a
whole chunk later, so the atomic's round trip is hidden.  ptxas likes to "aggregate" an atomic whose
addend is a constant or warp-uniform -- VOTE + FLO elect a lane, it adds popc(mask), a SHFL hands the
result round -- even when one lane is active, and that shuffle waits for the round trip on the spot (it
cost the step about 5 % when it happened).  spegg_fused.cuh prevents it with a
64-bit atomic whose addend is read back through shared memory; nothing but the SASS says whether the
trick still works after a toolkit update, so the SASS is what this test reads."""
import os
import re
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def sass():
    from paper_1603_09255_b200 import build
    so = build.build()
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(exe):
        pytest.skip("cuobjdump not available")
    txt = subprocess.run([exe, "-sass", so], check=True, capture_output=True, text=True).stdout
    funcs = {}
    name = None
    for line in txt.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            funcs[name] = []
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(.*?);", line)
        if m and name:
            funcs[name].append(m.group(1).strip())
    return funcs


def test_built_for_sm_100a_and_kernels_present(sass):
    names = "\n".join(sass)
    for k in ("k_fused_bit_f", "k_scan_fused", "k_fec_scan", "k_select_compact", "k_gamete_q10v", "k_offsets_static"):
        assert k in names, k


def test_ticket_atomic_of_the_fused_kernel_is_not_warp_aggregated(sass):
    fused = {n: ins for n, ins in sass.items() if "k_fused_bit_f" in n}
    assert len(fused) == 4                       # with / without the weighted father (MATE) x with / without residual noise (NOISE)
    for name, ins in fused.items():
        # the ticket: the only 64-bit global add whose old value is USED (destination register, not RZ)
        idx = [i for i, s in enumerate(ins) if re.search(r"ATOMG\.E\.ADD\.64\S* PT, R\d+,", s)]
        assert len(idx) == 1, (name, [ins[i] for i in idx])
        i = idx[0]
        # the aggregated form computes its addend in front of the atomic (elect a lane, count the others) and
        # consumes the result in a shuffle right behind it; here the atomic stands alone and the next thing
        # the warp does is the chunk's work
        for s in ins[max(0, i - 12):i]:
            assert not re.match(r"(@!?U?P\d+ )?(VOTE|VOTEU|FLO|UFLO|POPC|UPOPC|MATCH|REDUX)\b", s), (name, s)
        for s in ins[i + 1:i + 4]:
            assert not re.match(r"(@!?U?P\d+ )?SHFL\b", s), (name, s)
        # and its addend is a register loaded at run time, not an immediate
        assert re.search(r"\], R\d+$", ins[i].strip()), ins[i]


def test_recombination_carry_chain_is_the_probed_form(sass):
    """q10_push (sub.cc + addc) must compile to the carry-out of an IADD3 feeding an IMAD.X / IADD3.X --
    the same form in the hot kernels and in the create-time probe k_selftest_push, so that the probe tests
    what the kernels run."""
    probe = [ins for n, ins in sass.items() if "k_selftest_push" in n]
    assert len(probe) == 1
    assert sum(bool(re.search(r"IADD3 RZ, P\d", s)) for s in probe[0]) == 5
    assert sum(bool(re.search(r"(IMAD|IADD3)\.X ", s)) for s in probe[0]) >= 3       # (the first pushes fold into SEL)
    for n, ins in sass.items():
        if "k_gamete_q10v" in n or "k_gamete_q10r" in n:
            assert sum(bool(re.search(r"IADD3 RZ, P\d", s)) for s in ins) >= 8, n
            assert sum(bool(re.search(r"(IMAD|IADD3)\.X ", s)) for s in ins) >= 7, n
