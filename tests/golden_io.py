"""Reader for the small text fixtures under tests/golden/ (see its README)."""
import math
import os

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _num(expr):
    return float(eval(expr, {"__builtins__": {}}, {"sqrt": math.sqrt}))


def records(name):
    out = []
    with open(os.path.join(HERE, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                out.append([c.strip() for c in line.split("|")])
    return out


def numbers(field):
    return [_num(x) for x in field.split(",")]


number = _num
