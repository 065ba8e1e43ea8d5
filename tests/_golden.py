"""Parser for the small text fixtures under tests/golden/ (``key: value`` lines, ``#`` comments)."""
import os

_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def load(name):
    out = {}
    with open(os.path.join(_DIR, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, _, val = line.partition(":")
            out[key.strip()] = val.strip()
    return out


def ints(s):
    return [int(x) for x in s.split()]


def groups(s):
    """'0 1 | 2 | -' -> [[0,1],[2],[]]"""
    if not s.strip():
        return []
    return [[int(x) for x in part.split() if x != "-"] for part in s.split("|")]
