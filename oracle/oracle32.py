"""The oracle's fp32 re-run mode (SURVEY 8(c) reading 23).  TEST INFRASTRUCTURE ONLY, like oracle.py.

The same ctypes front-end (oracle/oracle.py, executed a second time with _ORACLE_FP32 set) over liboracle32.so: the
same C source compiled with every `double` a `float`, libm's single-precision functions and single-precision
literals.  Its only use is to print the fp32 NOISE FLOOR -- how far a careful fp32 implementation of the oracle's own
formulas lands from the fp64 oracle -- next to each parity tolerance (tests/test_oracle_fp32_floor.py); the GPU path is
never compared with it.  Usage:  from oracle import oracle32;  oracle32.iteration(p, ...)  (every function of
oracle.oracle, arrays come back as float32)."""
import os
import sys
import types

_HERE = os.path.dirname(os.path.abspath(__file__))
_mod = types.ModuleType("oracle._oracle_fp32")
_mod.__file__ = os.path.join(_HERE, "oracle.py")
_mod.__dict__["_ORACLE_FP32"] = True
with open(_mod.__file__) as _f:
    exec(compile(_f.read(), _mod.__file__, "exec"), _mod.__dict__)
sys.modules[_mod.__name__] = _mod

for _name, _value in list(_mod.__dict__.items()):
    if not _name.startswith("__"):
        globals()[_name] = _value
