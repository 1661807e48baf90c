"""paper_2607_04676_b200 - B200-native (sm_100a) Pici hot path of SpCCL's sparse collectives.

`pici`  : ctypes binding of the C-ABI library libpici_b200 (include/pici.h)
`ring`  : host driver running ring all-gather / reduce-scatter / all-reduce over P logical ranks in one HBM
`build` : nvcc build of the in-tree shared library
"""
from . import build, pici  # noqa: F401
