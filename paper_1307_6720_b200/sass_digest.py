"""SASS digest of the hot kernels of libmhs_b200.so: registers / shared memory per kernel (cuobjdump -res-usage) and an opcode
histogram with the bulk-copy / mbarrier instructions that prove the sm_100a data path (UBLKCP = cp.async.bulk, SYNCS = mbarrier).

    python -m paper_1307_6720_b200.sass_digest [regex of demangled kernel names]  > profiles/rNN_sass_digest.md

Runs on the CPU box (no GPU needed); it reads the in-tree .so that `python -m paper_1307_6720_b200.build` made."""
from __future__ import annotations

import collections
import re
import subprocess
import sys

from . import build as _build

DEFAULT = r"k_zsweep<double, 4, 2, 0, 0, (1, 0|0, 1), 1>|k_resid_restrict_ring<double>|k_fields_ring<double, 256|k_resid_restrict_sep<double, 4, 0>|k_fields_z<double|k_zline<double, 0>|k_fieldlines<double>|k_cluster<double, [01]>|k_resnorm_static_partial<double>"


def demangle(names):
    out = subprocess.run(["cu++filt"] + names, capture_output=True, text=True).stdout.splitlines()
    return [o.strip() for o in out]


def main(pattern=DEFAULT):
    lib = _build.LIB
    rx = re.compile(pattern)
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True).stdout
    res = subprocess.run(["cuobjdump", "-res-usage", lib], capture_output=True, text=True).stdout
    usage = {}
    cur = None
    for line in res.splitlines():
        m = re.search(r"Function (\S+):", line)
        if m:
            cur = m.group(1)
            continue
        if cur and "REG:" in line:
            usage[cur] = line.strip()
            cur = None
    hist = collections.OrderedDict()
    cur = None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            hist[cur] = collections.Counter()
            continue
        m = re.match(r"\s+/\*[0-9a-f]+\*/\s+(@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]+)", line)
        if cur and m:
            op = m.group(2)
            key = op if op.startswith(("UBLKCP", "SYNCS", "LDS", "STS", "LDG", "STG", "UTMA", "BAR", "ACQBULK")) else op.split(".")[0]
            hist[cur][key] += 1
    names = list(hist)
    dem = dict(zip(names, demangle(names)))
    print("# SASS digest of %s\n" % lib.split("/")[-1])
    print("Command: `python -m paper_1307_6720_b200.sass_digest` (cuobjdump -sass / -res-usage of the in-tree library; static counts, whole kernel).\n")
    for n in names:
        d = re.sub(r"\((int|bool)\)", "", dem.get(n, n))      # cu++filt writes template arguments as (int)4, (bool)0
        if not rx.search(d):
            continue
        h = hist[n]
        tot = sum(h.values())
        print("## `%s`\n" % d.replace("mhs::", ""))
        print("%s; %d SASS instructions\n" % (usage.get(n, "?"), tot))
        print("| opcode | count | opcode | count | opcode | count |")
        print("|---|---|---|---|---|---|")
        items = h.most_common(24)
        for i in range(0, len(items), 3):
            row = items[i:i + 3] + [("", "")] * (3 - len(items[i:i + 3]))
            print("| " + " | ".join("%s | %s" % (a, b) for a, b in row) + " |")
        special = {k: v for k, v in h.items() if k.startswith(("UBLKCP", "SYNCS", "UTMA"))}
        print("\nbulk-copy / mbarrier instructions: %s\n" % (", ".join("%s x%d" % kv for kv in sorted(special.items())) or "none"))


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else DEFAULT)
