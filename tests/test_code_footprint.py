"""Guard on the instruction footprint of the dual-lane attention kernel (no GPU: reads the SASS of the
built libcp.so with cuobjdump).

DESIGN.md 7.0: seven warp roles of `dl::attn_dl_kernel` run different code at once against the SM's 32 KB
L1.5 instruction cache; at 19,216 SASS instructions (a `producer` copy per lane, runtime divisions by the
GQA group size in column-unrolled code) a mixed batch spent 27 % of its issue slots waiting for instruction
fetch and ran 1.4x slower.  The kernel was 14,560 instructions after that fix; this test fails if it grows back.
Round 2 added ~600 instructions per softmax role for the in-kernel merge of split decode groups: it
runs once per group, outside every per-tile loop, and the A/B on configs[2] showed no change -- the budgets below
leave room for exactly that and nothing else.  The fp8 instantiation went from 11,760 to 7,928 instructions when its
two softmax warpgroups began to share one code copy (512 decodes over fp8 pages 334 -> 296 us).
"""
import re
import shutil
import subprocess

import pytest

from paper_2606_09061_b200 import build

# instantiation (D, POLY, SPLIT, KV8, APPEND) -> budget in SASS instructions
BUDGET = {"ILi128ELb0ELb0ELb0ELb0E": 15900,      # dual lane, bf16 pages: the HBM-bound mixed batch (the bench workload)
          "ILi128ELb0ELb0ELb0ELb1E": 14600,      # the same with H2 inside (small decode-only batches: no tile items run, its tile code is cold)
          "ILi128ELb1ELb1ELb0ELb0E": 11500,      # SPLIT: tensor-bound batches
          "ILi128ELb0ELb0ELb1ELb0E": 8100,       # dual lane over fp8 (e4m3) pages: ONE softmax code copy for both warpgroups
          "ILi64ELb0ELb0ELb0ELb0E": 4200, "ILi64ELb1ELb1ELb0ELb0E": 5400}


@pytest.mark.skipif(shutil.which("cuobjdump") is None, reason="cuobjdump not on PATH")
def test_dual_lane_kernel_sass_size_within_budget():
    lib = build.build()
    sass = subprocess.run(["cuobjdump", "-sass", lib], check=True, capture_output=True, text=True).stdout
    counts, cur = {}, None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            continue
        if cur and re.match(r"\s+/\*[0-9a-f]{4,5}\*/\s+\S", line):
            counts[cur] = counts.get(cur, 0) + 1
    kernels = {k: v for k, v in counts.items() if "attn_dl_kernel" in k}
    assert len(kernels) == len(BUDGET), list(kernels)
    for key, limit in BUDGET.items():
        hits = {k: v for k, v in kernels.items() if "attn_dl_kernel" + key in k}
        assert len(hits) == 1, (key, list(kernels))
        for name, n in hits.items():
            assert 1000 < n <= limit, f"{name}: {n} SASS instructions > budget {limit} (DESIGN.md 7.0)"
    # a runtime integer division shows up as a reciprocal sequence starting with I2F.U32.RP
    for body in sass.split("attn_dl_kernelILi128ELb0ELb0ELb0ELb0E")[1:]:
        assert body.split("Function :", 1)[0].count("I2F.U32.RP") <= 4, "runtime integer divisions crept back"


@pytest.mark.skipif(shutil.which("cuobjdump") is None, reason="cuobjdump not on PATH")
def test_attention_kernel_is_blackwell_native():
    """The SASS of every attention-kernel instantiation holds tcgen05 MMAs (UTCHMMA), TMEM loads / stores
    (LDTM / STTM) and TMA loads (UTMALDG), and no legacy tensor path (HMMA = mma.sync / wmma).  Counts are
    committed under profiles/ (r02_sass_mnemonics.md)."""
    lib = build.build()
    sass = subprocess.run(["cuobjdump", "-sass", lib], check=True, capture_output=True, text=True).stdout
    bodies = {}
    for part in sass.split("Function : ")[1:]:
        name, body = part.split("\n", 1)
        bodies[name.strip()] = body
    kernels = {k: v for k, v in bodies.items() if "attn_dl_kernel" in k}
    assert len(kernels) >= 4
    for name, body in kernels.items():
        if "ELb1ELb0EEEv" in name:               # KV8
            assert body.count("UTCQMMA") > 0, f"{name}: no fp8 tcgen05.mma (UTCQMMA) in the SASS"
        for mnemonic in ("UTCHMMA", "LDTM", "STTM", "UTMALDG", "UTCBAR"):
            assert body.count(mnemonic) > 0, f"{name}: no {mnemonic} in the SASS"
        assert not re.search(r"\bHMMA\b", body), f"{name}: legacy mma.sync path present"
    assert not any("attn_simt" in k or "attn_tc" in k for k in bodies), "debug-only kernels in the shipped library"
