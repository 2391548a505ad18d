"""The pair kernel's tile feed frees a slot with a RELAXED remote arrive whose address carries a register dependency on the
value just loaded from that slot (csrc/ptx.cuh, mbar_arrive_cluster_after).  Round 1's form of that dependency (`dep & 0`)
was folded away by ptxas and the arrive overtook the load (profiles/r2_feed_race.md).  This test reads the SASS of the built
library and checks that the dependency is still there: in every xengine_pair_kernel instantiation the three feed readers
(TMA producer, MMA issuer, epilogue warps) each compute the arrive's address as `LEA.HI Rd, Rloaded, Rbase, RZ, 0x1`
(= Rbase + (Rloaded >> 31)) from a register an LDS wrote, and use Rd as the address of a SYNCS.ARRIVE shortly after.
A toolchain update that folds it again fails here, without needing a GPU.
"""
import re
import shutil
import subprocess

import pytest


def _functions(sass):
    name, body = None, []
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            if name:
                yield name, body
            name, body = m.group(1), []
        else:
            m = re.match(r"\s+/\*[0-9a-f]+\*/\s+(.*?);", line)
            if m and name:
                body.append(m.group(1).strip())
    if name:
        yield name, body


def test_feed_arrive_address_depends_on_the_slot_load():
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not shutil.which(cuobjdump):
        pytest.skip("cuobjdump not available")
    from paper_1305_5639_b200 import binding
    binding.lib()
    sass = subprocess.run([cuobjdump, "-sass", binding.LIB_PATH], capture_output=True, text=True, check=True).stdout
    seen = 0
    for name, ins in _functions(sass):
        if "xengine_pair_kernel" not in name:
            continue
        seen += 1
        chains = 0
        for k, text in enumerate(ins):
            m = re.search(r"LEA\.HI (R\d+), (R\d+), (R\d+), RZ, 0x1\b", text)
            if not m:
                continue
            rd, rs = m.group(1), m.group(2)
            # (the compiler moves the divergent copies of these sequences out of line, far from the load: the source register
            # only has to be one an LDS writes somewhere in the kernel; the arrive follows within a few instructions)
            loaded = any(re.search(r"\bLDS(\.\w+)* %s," % rs, t) for t in ins)
            used = any(re.search(r"SYNCS\.ARRIVE\S* RZ, \[%s\+" % rd, t) for t in ins[k + 1:k + 12])
            chains += bool(loaded and used)
        assert chains >= 3, "%s: only %d load -> address -> remote-arrive chains left in the SASS" % (name, chains)
    assert seen == 2, "expected the int8 and the fp16 instantiation of the pair kernel, found %d" % seen
