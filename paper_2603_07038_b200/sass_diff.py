"""Kernel-by-kernel comparison of two builds of libem.so (beside build.py: the check behind "this change left the measured
kernels alone").  python -m paper_2603_07038_b200.sass_diff OLD.so NEW.so

For every kernel present in both libraries: `identical`, `parameter offsets only` (the same instruction stream, only
c[0x0][..] kernel-parameter offsets moved because a parameter struct grew) or `changed` (with the instruction counts)."""
from __future__ import annotations

import functools
import re
import subprocess
import sys


@functools.lru_cache(maxsize=4)
def kernels(lib: str) -> dict[str, list[str]]:
    out = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    mangled = re.findall(r"Function : (\S+)", out)
    names = subprocess.run(["c++filt"], input="\n".join(mangled), capture_output=True, text=True, check=True).stdout.split("\n")
    d: dict[str, list[str]] = {}
    cur = None
    it = iter(names)
    for line in out.splitlines():
        if re.match(r"\s*Function : ", line):
            cur = next(it).split("(")[0]
            d[cur] = []
        elif cur is not None and re.search(r"/\*[0-9a-f]{4}\*/", line):
            s = re.sub(r"/\*[0-9a-f]{4}\*/", "", line)
            d[cur].append(re.sub(r"/\* 0x[0-9a-f]+ \*/", "", s).strip())
    return d


def compare(old: str, new: str) -> dict[str, str]:
    a, b = kernels(old), kernels(new)
    strip = lambda L: [re.sub(r"c\[0x0\]\[0x[0-9a-f]+\]", "c[P]", x) for x in L]
    res = {}
    for k in sorted(set(a) | set(b)):
        if k not in a:
            res[k] = "new"
        elif k not in b:
            res[k] = "removed"
        elif a[k] == b[k]:
            res[k] = "identical"
        elif strip(a[k]) == strip(b[k]):
            res[k] = "parameter offsets only"
        else:
            res[k] = f"changed ({len(a[k])} -> {len(b[k])} instructions)"
    return res


if __name__ == "__main__":
    for k, v in compare(sys.argv[1], sys.argv[2]).items():
        print(f"{v:36s} {k}")
