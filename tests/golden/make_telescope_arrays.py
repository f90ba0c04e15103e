#!/usr/bin/env python
"""Extract the two model telescope arrays the thesis prints (Appendix B.3)
into small text fixtures, so that tests can run where /root/reference does not exist.

    python tests/golden/make_telescope_arrays.py [/root/reference/PAPER.md]

Array 1 (B.3.2): 13 telescopes, columns x, y, z, radius [m].  The PDF extraction shifted
the columns one to the left (the ID column holds x, ..., the "z" column holds the radius, the last
column is empty); the parser reads the four numbers of each row in order.
Array 2 (B.3.3 Table B.1): 180 telescopes, two per table row as
"ID | x, y, z | radius m".
Nothing is retyped: every number is parsed from PAPER.md.
"""
import os
import re
import sys

HERE = os.path.dirname(os.path.abspath(__file__))


def parse(paper_path: str):
    lines = open(paper_path, encoding="utf-8").read().split("\n")
    i1 = next(i for i, l in enumerate(lines) if "B.3.2" in l and "Telescope Array 1" in l and l.startswith("#"))
    i2 = next(i for i, l in enumerate(lines) if "B.3.3" in l and "Telescope Array 2" in l and l.startswith("#"))
    num = r"-\s*\d+(?:\.\d+)?|\d+(?:\.\d+)?"
    arr1 = []
    for l in lines[i1:i2]:
        if not l.startswith("|") or "---" in l or "ID" in l:
            continue
        vals = [float(v.replace(" ", "")) for v in re.findall(num, l)]
        if len(vals) == 4:
            arr1.append(vals)
    arr2 = {}
    pat = re.compile(r"\|\s*(\d+)\s*\|\s*(" + num + r")\s*,\s*(" + num + r")\s*,\s*(" + num + r")\s*\|\s*(\d+(?:\.\d+)?)\s*m")
    for l in lines[i2:]:
        if l.startswith("#") and "B.3.3" not in l:
            break
        for m in pat.finditer(l):
            arr2[int(m.group(1))] = [float(m.group(k).replace(" ", "")) for k in (2, 3, 4, 5)]
    return arr1, [arr2[k] for k in sorted(arr2)], (i1 + 1, i2 + 1)


def write(name, rows, cite):
    with open(os.path.join(HERE, name), "w") as f:
        f.write(f"# {cite}\n# x[m] y[m] z[m] radius[m]\n")
        for r in rows:
            f.write(" ".join(f"{v:g}" for v in r) + "\n")


if __name__ == "__main__":
    paper = sys.argv[1] if len(sys.argv) > 1 else "/root/reference/PAPER.md"
    a1, a2, (l1, l2) = parse(paper)
    assert len(a1) == 13 and len(a2) == 180, (len(a1), len(a2))
    write("telescope_array_1.txt", a1, f"thesis Appendix B.3.2 'Telescope Array 1' (PAPER.md line {l1} ff.), parsed by make_telescope_arrays.py")
    write("telescope_array_2.txt", a2, f"thesis Appendix B.3.3 'Telescope Array 2', Table B.1 (PAPER.md line {l2} ff.), parsed by make_telescope_arrays.py")
    print(len(a1), len(a2))
