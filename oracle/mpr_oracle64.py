"""The CPU oracle with double storage of data and state (the paper's double-precision program, Table 2;
SURVEY 8(f) NEXT-3): the same C source built with -DORC_F64 and the same wrapper bound to float64 arrays.

A second instance of the module oracle/mpr_oracle.py, made by the import machinery with `_F64 = True` set in the new
module before its body runs (the body reads it to pick the storage type and the library to build); the names of
that instance are re-exported here.

TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/mpr_oracle.py)."""
import importlib.util as _util
import os as _os
import sys as _sys

_spec = _util.spec_from_file_location(
    "oracle._mpr_oracle_f64", _os.path.join(_os.path.dirname(_os.path.abspath(__file__)), "mpr_oracle.py"))
_impl = _util.module_from_spec(_spec)
_impl._F64 = True
_sys.modules[_spec.name] = _impl          # dataclasses looks its module up by name while the body runs
_spec.loader.exec_module(_impl)
globals().update({_k: _v for _k, _v in vars(_impl).items() if not _k.startswith("__")})
