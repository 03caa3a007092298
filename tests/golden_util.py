"""Reader for tests/golden/*.txt (`key = value` lines, optional [sections], `#` comments)."""
import os

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_golden(name):
    out, sec = {}, None
    with open(os.path.join(GOLDEN, name)) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            if line.startswith("[") and line.endswith("]"):
                sec = line[1:-1]
                out[sec] = {}
                continue
            k, v = (s.strip() for s in line.split("=", 1))
            (out[sec] if sec else out)[k] = v
    return out


def num(v):
    try:
        return int(v)
    except ValueError:
        return float(v)
