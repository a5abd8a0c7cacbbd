"""The CPU oracle with double storage of data and state (the paper's double-precision program, Table 2;
SURVEY 8(f) NEXT-3): the same C source built with -DORC_F64 and the same wrapper bound to float64 arrays.

TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/mpr_oracle.py)."""
import os as _os

_path = _os.path.join(_os.path.dirname(_os.path.abspath(__file__)), "mpr_oracle.py")
_F64 = True
with open(_path) as _f:
    exec(compile(_f.read(), _path, "exec"), globals())
