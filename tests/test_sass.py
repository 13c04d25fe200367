"""Static check of the built library (no GPU): the hot loop of the shared-memory traversal.

DESIGN.md 6.1 / 6.2: two lines per trip in 15 SASS instructions (2 DADD, 2 x [SHF, LEA/IMAD, 2 LDS, SHF.W], LOP3,
ISETP, BRA).  ptxas has twice turned it into 19 (extra MOVs; the exponent offset re-added per address) when the
surrounding code changed, which costs the whole kernel ~12 %: this test pins the count in every kernel that
inlines cast_beam_smem."""
import os
import re
import shutil
import subprocess

import pytest


def _cuobjdump():
    for c in (shutil.which("cuobjdump"), "/usr/local/cuda/bin/cuobjdump"):
        if c and os.path.exists(c):
            return c
    return None


def test_hot_loop_is_15_instructions_in_every_kernel():
    exe = _cuobjdump()
    if exe is None:
        pytest.skip("cuobjdump not found")
    from paper_2606_15846_b200 import build
    build.build()
    sass = subprocess.run([exe, "-sass", build.LIB], capture_output=True, text=True, check=True).stdout
    found = {}
    for f in re.split(r"\n\s*Function : ", sass)[1:]:
        name = f.split("\n")[0]
        addr, ins = [], []
        for line in f.split("\n"):
            m = re.search(r"/\*([0-9a-f]{4,5})\*/\s+(.*?);", line)
            if m:
                addr.append(int(m.group(1), 16))
                ins.append(m.group(2))
        for i, t in enumerate(ins):
            m = re.search(r"BRA.*?(0x[0-9a-f]+)", t)
            if not m:
                continue
            tgt = int(m.group(1), 16)
            if tgt < addr[i] and addr[i] - tgt < 0x200 and tgt in addr:
                body = ins[addr.index(tgt):i + 1]
                # the paired-line loop: exactly two DADD (the two crossings) and four LDS (two windows)
                if sum("LDS" in b for b in body) == 4 and sum("DADD" in b for b in body) == 2:
                    found[name] = len(body)
    kernels = [k for k in found if "beam_kernel" in k]
    # the production kernels: beam_kernel<smem, !aux>, step_beam_kernel<smem, !aux>, reset_beam_kernel<!aux>
    assert len(kernels) >= 3, found
    for k in kernels:
        assert found[k] == 15, (k, found[k])
