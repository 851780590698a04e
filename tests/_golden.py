"""Readers for tests/golden/*.txt (paper-printed values and cited fixtures)."""
import os

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_pins(name="paper_pins.txt"):
    pins = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) == 2:
                pins[line[0]] = float(line[1]) if "." in line[1] else int(line[1])
    return pins


def read_whole_maps():
    maps = {}
    with open(os.path.join(GOLDEN, "whole_maps.txt")) as f:
        for line in f:
            t = line.split("#")[0].split()
            if len(t) < 9:
                continue
            num = lambda s: None if s == "-" else int(s)
            maps[t[0]] = dict(N=int(t[1]), folding=int(t[2]), null=int(t[3]), top5=[int(x) for x in t[4].split(",")],
                              sumR=int(t[5]), sumD=int(t[6]), sumO=int(t[7]), pairs=int(t[8]),
                              nn_total=num(t[9]), nn_one=num(t[10]), nn_max=num(t[11]))
    return maps


def read_3x3_fixture():
    fx = dict(structures=[], genotypes=[])
    with open(os.path.join(GOLDEN, "lattice_3x3.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if not line:
                continue
            tag, rest = line[0], line[1:]
            parts = [p.split() for p in rest.split("|")]
            if tag == "S":
                fx["structures"].append(dict(d=int(parts[0][0]), sites=[int(x) for x in parts[1]], cls=int(parts[2][0]),
                                             contacts=[tuple(int(v) for v in c.split("-")) for c in parts[3]]))
            elif tag == "G":
                fx["genotypes"].append(dict(g=int(parts[0][0]), energies=[int(x) for x in parts[1]],
                                            pheno=None if parts[2][0] == "NULL" else int(parts[2][0])))
            elif tag == "H":
                fx["hist"] = [int(x) for x in parts[0]]
                fx["null"] = int(parts[1][0])
            else:
                fx[tag] = [int(x) for x in parts[0]]
    return fx
