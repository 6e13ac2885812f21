"""ORACLE (test infrastructure): builds and loads the oracle's C core with gcc.

``gcc -O2 -ffp-contract=off -fopenmp``: no fused multiply-add, so the float64
expression order in ``zda_oracle_core.c`` is what is evaluated.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "zda_oracle_core.c")
_LIB = os.path.join(_HERE, "libzda_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    objs = []
    for tag, defs in (("re", []), ("cx", ["-DZO_COMPLEX"])):
        obj = os.path.join(_HERE, f"zda_oracle_core_{tag}.o")
        subprocess.check_call(["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC",
                               "-Wall", "-c", _SRC, "-o", obj] + defs)
        objs.append(obj)
    subprocess.check_call(["gcc", "-shared", "-fopenmp", "-o", _LIB] + objs + ["-lm"])
    for o in objs:
        os.remove(o)
    return _LIB


def load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
    return _lib
