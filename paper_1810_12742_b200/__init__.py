"""paper_1810_12742_b200 -- thin Python binding of libhines_b200.so (include/hines.h).

Argument marshalling only: every step of the solve runs in the library's CUDA kernels.
PyTorch is used by callers for device memory and streams; this module passes raw pointers.
There is no CPU fallback: if the extension is missing or there is no GPU, calls fail loudly.

Names mirror the C ABI: hines_plan_create -> Plan(...), hines_solve -> Plan.solve,
hines_solve_host -> Plan.solve_host, hines_plan_get_info -> Plan.info,
hines_plan_get_table -> Plan.table, hines_plan_destroy -> Plan.close.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from ._build import LIB as _LIB_PATH, build as build_library

F64, F32 = 0, 1
POLICY_DEFAULT, POLICY_FORCE_STREAM, POLICY_NO_GROUPING, POLICY_INPUT_ORDER, POLICY_NO_CLUSTER = 0, 1, 2, 4, 8
POLICY_SERIAL_CLASSES = 16
POLICY_POW2_CLUSTERS = 32
POLICY_NO_SPLIT = 64
POLICY_SPLIT_LEVEL_MEAN = 128
POLICY_NO_PCR = 256
POLICY_FACTORED = 512
POLICY_NO_QUADS = 1024
POLICY_NO_PDL = 2048
POLICY_SPLIT_BLOCK_MEAN = 4096
ITEM_SINGLE, ITEM_CLUSTER, ITEM_SPLIT = 0, 1, 2

STATUS = {0: "HINES_OK", 1: "HINES_ERR_INVALID_ARG", 2: "HINES_ERR_BAD_TOPOLOGY", 3: "HINES_ERR_ALLOC",
          4: "HINES_ERR_CUDA", 5: "HINES_ERR_UNSUPPORTED"}

# table id -> (name, numpy dtype)
TABLES = {
    "cell_branch_offsets": (0, np.int64), "branch_start": (1, np.int32), "branch_len": (2, np.int32),
    "branch_parent_comp": (3, np.int32), "branch_parent_branch": (4, np.int32), "branch_level": (5, np.int32),
    "cell_nlevels": (6, np.int32), "cell_level_offsets": (7, np.int64), "level_count": (8, np.int32),
    "level_list": (9, np.int32), "child_offsets": (10, np.int64), "child_ids": (11, np.int32),
    "cell_item": (32, np.int32), "item_cell_offsets": (33, np.int64), "item_cells": (37, np.int64), "item_class": (34, np.int32),
    "item_launch_order": (35, np.int32), "item_kind": (36, np.int32), "item_xch": (44, np.int32),
    "item_part_offsets": (46, np.int64), "part_header": (47, np.int32), "part_meta": (48, np.int32),
    "part_runs": (49, np.int32),
    "stream_level_begin": (40, np.int64), "stream_desc": (41, np.int32), "stream_child": (42, np.int32),
    "class_smem_bytes": (43, np.int32), "class_cluster": (50, np.int32), "class_threads": (51, np.int32),
    "class_phase": (52, np.int32), "class_first": (53, np.int64), "class_count": (54, np.int64),
    "class_parts": (55, np.int32),
    "split_piece_offsets": (60, np.int64), "split_piece_len": (61, np.int32), "split_piece_level": (62, np.int32),
    "split_level_stat": (63, np.int64),
}

# every symbol include/hines.h declares
ABI_SYMBOLS = ["hines_plan_create", "hines_partition_cells", "hines_reroot", "hines_gather", "hines_scatter", "hines_factor", "hines_solve_rhs", "hines_plan_upload", "hines_solve", "hines_solve_host", "hines_solve_static",
               "hines_host_pipeline_create", "hines_host_pipeline_solve", "hines_host_pipeline_slices", "hines_host_pipeline_destroy",
               "hines_plan_destroy", "hines_plan_get_info", "hines_plan_get_table",
               "hines_plan_launches_per_solve", "hines_plan_enable_timing", "hines_plan_get_timing",
               "hines_plan_enable_phase_clocks", "hines_plan_get_phase_clocks",
               "hines_status_string", "hines_last_error", "hines_version"]


class Options(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("threads_per_block", C.c_int32),
                ("smem_bytes_per_block", C.c_int32), ("policy_flags", C.c_int32),
                ("stream_threads", C.c_int32), ("group_smem_bytes", C.c_int32), ("max_segment", C.c_int32),
                ("cluster_max", C.c_int32), ("chunk_smem_bytes", C.c_int32), ("split_smem_bytes", C.c_int32)]


class PlanInfo(C.Structure):
    _fields_ = [("n", C.c_int64), ("ncells", C.c_int64), ("nbranches", C.c_int64),
                ("max_levels", C.c_int32), ("dtype", C.c_int32),
                ("n_resident_items", C.c_int64), ("n_resident_cells", C.c_int64),
                ("n_resident_unknowns", C.c_int64), ("n_stream_cells", C.c_int64),
                ("n_stream_unknowns", C.c_int64), ("n_stream_branches", C.c_int64),
                ("padded_lane_steps", C.c_int64), ("useful_lane_steps", C.c_int64),
                ("workspace_bytes", C.c_int64), ("bytes_min", C.c_int64), ("bytes_literal", C.c_int64),
                ("breadth_first", C.c_int32), ("n_classes", C.c_int32),
                ("n_cluster_cells", C.c_int64), ("n_cluster_unknowns", C.c_int64), ("n_parts", C.c_int64),
                ("n_split_cells", C.c_int64), ("n_split_unknowns", C.c_int64), ("n_exports", C.c_int64),
                ("n_blocks", C.c_int64)]


class HinesError(RuntimeError):
    def __init__(self, status, detail):
        super().__init__(f"{STATUS.get(status, status)}: {detail}")
        self.status = status


_lib = None


def load_library(build_if_missing: bool = True):
    """dlopen libhines_b200.so (built in-tree).  Raises if it cannot be found or built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        if not build_if_missing:
            raise ImportError(f"{_LIB_PATH} missing: run `python -c 'import __graft_entry__ as g; g.build()'`")
        build_library()
    lib = C.CDLL(_LIB_PATH)
    vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int32
    lib.hines_plan_create.argtypes = [vp, vp, i64, i32, C.POINTER(Options), C.POINTER(vp)]
    lib.hines_plan_upload.argtypes = [vp]
    lib.hines_partition_cells.argtypes = [vp, i64, i32, vp, vp]
    lib.hines_reroot.argtypes = [vp, vp, i64, vp, vp, vp, vp, vp, vp]
    lib.hines_gather.argtypes = [vp, vp, vp, i64, i32, vp]
    lib.hines_scatter.argtypes = [vp, vp, vp, i64, i32, vp]
    lib.hines_solve.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.hines_solve_host.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.hines_solve_static.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp, i32, vp]
    lib.hines_host_pipeline_create.argtypes = [vp, vp, i64, i32, C.POINTER(Options), i32, C.POINTER(vp)]
    lib.hines_host_pipeline_solve.argtypes = [vp, vp, vp, vp, vp]
    lib.hines_host_pipeline_slices.argtypes = [vp, C.POINTER(i32), vp, i64]
    lib.hines_host_pipeline_destroy.argtypes = [vp]
    lib.hines_factor.argtypes = [vp, vp, vp, vp]
    lib.hines_solve_rhs.argtypes = [vp, vp, vp, vp]
    lib.hines_plan_destroy.argtypes = [vp]
    lib.hines_plan_get_info.argtypes = [vp, C.POINTER(PlanInfo)]
    lib.hines_plan_get_table.argtypes = [vp, i32, vp, i64, C.POINTER(i64)]
    lib.hines_plan_launches_per_solve.argtypes = [vp, C.POINTER(i32)]
    lib.hines_plan_enable_timing.argtypes = [vp, i32]
    lib.hines_plan_get_timing.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_float)]
    lib.hines_plan_enable_phase_clocks.argtypes = [vp, i32]
    lib.hines_plan_get_phase_clocks.argtypes = [vp, vp, i64, C.POINTER(i64)]
    for f in ("hines_status_string", "hines_last_error", "hines_version"):
        getattr(lib, f).restype = C.c_char_p
    lib.hines_status_string.argtypes = [i32]
    _lib = lib
    return lib


def _check(status):
    if status != 0:
        raise HinesError(status, load_library().hines_last_error().decode())


def _ptr(t):
    """Raw address of a torch tensor / numpy array / int."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    assert t.is_contiguous()
    return t.data_ptr()


class Plan:
    """hines_plan_create(parent arrays, cell offsets) -- setup-time scheduler."""

    def __init__(self, parent, cell_offsets, dtype=F64, threads_per_block=0, smem_bytes_per_block=0,
                 policy_flags=0, stream_threads=0, group_smem_bytes=0, max_segment=0, cluster_max=0,
                 chunk_smem_bytes=0, split_smem_bytes=0):
        lib = load_library()
        parent = np.ascontiguousarray(parent, dtype=np.int32)
        offs = np.ascontiguousarray(cell_offsets, dtype=np.int64)
        opt = Options(C.sizeof(Options), threads_per_block, smem_bytes_per_block, policy_flags,
                      stream_threads, group_smem_bytes, max_segment, cluster_max, chunk_smem_bytes, split_smem_bytes)
        h = C.c_void_p()
        self._h = None
        _check(lib.hines_plan_create(parent.ctypes.data, offs.ctypes.data, len(offs) - 1, int(dtype),
                                     C.byref(opt), C.byref(h)))
        self._h = h
        self.dtype = int(dtype)
        self.np_dtype = np.float64 if self.dtype == F64 else np.float32

    # hines_plan_get_info
    @property
    def info(self) -> PlanInfo:
        out = PlanInfo()
        _check(load_library().hines_plan_get_info(self._h, C.byref(out)))
        return out

    # hines_plan_get_table
    def table(self, name: str) -> np.ndarray:
        tid, dt = TABLES[name]
        need = C.c_int64()
        _check(load_library().hines_plan_get_table(self._h, tid, None, 0, C.byref(need)))
        out = np.empty(need.value // np.dtype(dt).itemsize, dtype=dt)
        _check(load_library().hines_plan_get_table(self._h, tid, out.ctypes.data, need.value, C.byref(need)))
        return out

    @property
    def launches_per_solve(self) -> int:
        out = C.c_int32()
        _check(load_library().hines_plan_launches_per_solve(self._h, C.byref(out)))
        return out.value

    # hines_plan_enable_timing / hines_plan_get_timing
    def enable_timing(self, enable=True):
        _check(load_library().hines_plan_enable_timing(self._h, int(bool(enable))))

    def timing(self):
        """(resident_ms, stream_ms) of the last solve; waits for it."""
        a, b = C.c_float(), C.c_float()
        _check(load_library().hines_plan_get_timing(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    # hines_plan_enable_phase_clocks / hines_plan_get_phase_clocks
    def enable_phase_clocks(self, enable=True):
        _check(load_library().hines_plan_enable_phase_clocks(self._h, int(bool(enable))))

    def phase_clocks(self) -> np.ndarray:
        """uint64[nblocks, 8] of the last solve (launch order); waits for the device."""
        need = C.c_int64()
        _check(load_library().hines_plan_get_phase_clocks(self._h, None, 0, C.byref(need)))
        out = np.zeros(need.value // 8, dtype=np.uint64)
        _check(load_library().hines_plan_get_phase_clocks(self._h, out.ctypes.data, need.value, C.byref(need)))
        return out.reshape(-1, 8)

    def upload(self):
        _check(load_library().hines_plan_upload(self._h))

    # hines_solve: device pointers (torch CUDA tensors or raw addresses); enqueues on `stream`
    def solve(self, d, u, b, x, stream=None):
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        _check(load_library().hines_solve(self._h, _ptr(d), _ptr(u), _ptr(b), _ptr(x), stream))
        return x

    # hines_factor / hines_solve_rhs (f3; plan created with POLICY_FACTORED)
    def factor(self, d, u, stream=None):
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        _check(load_library().hines_factor(self._h, _ptr(d), _ptr(u), stream))

    def solve_rhs(self, b, x, stream=None):
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        _check(load_library().hines_solve_rhs(self._h, _ptr(b), _ptr(x), stream))
        return x

    # hines_solve_host: host buffers (numpy arrays or pinned torch CPU tensors); synchronous
    def solve_host(self, d, u, b, x, stream=None):
        _check(load_library().hines_solve_host(self._h, _ptr(d), _ptr(u), _ptr(b), _ptr(x), stream or 0))
        return x

    def close(self):
        if self._h is not None:
            load_library().hines_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class HostPipeline:
    """hines_host_pipeline_*: host buffers in, host buffers out, the batch cut into slices of whole cells whose copy-in,
    solve and copy-out overlap (the end-to-end entry; options as for Plan)."""

    def __init__(self, parent, cell_offsets, dtype=F64, nslices=0, **options):
        lib = load_library()
        parent = np.ascontiguousarray(parent, dtype=np.int32)
        offs = np.ascontiguousarray(cell_offsets, dtype=np.int64)
        o = dict(threads_per_block=0, smem_bytes_per_block=0, policy_flags=0, stream_threads=0, group_smem_bytes=0,
                 max_segment=0, cluster_max=0, chunk_smem_bytes=0, split_smem_bytes=0)
        o.update(options)
        opt = Options(C.sizeof(Options), *[o[k] for k in ("threads_per_block", "smem_bytes_per_block", "policy_flags",
                                                           "stream_threads", "group_smem_bytes", "max_segment", "cluster_max",
                                                           "chunk_smem_bytes", "split_smem_bytes")])
        h = C.c_void_p()
        self._h = None
        _check(lib.hines_host_pipeline_create(parent.ctypes.data, offs.ctypes.data, len(offs) - 1, int(dtype), C.byref(opt),
                                              int(nslices), C.byref(h)))
        self._h = h
        self.dtype = int(dtype)

    def solve(self, d, u, b, x):
        """HOST buffers (numpy arrays or pinned torch CPU tensors); synchronous."""
        _check(load_library().hines_host_pipeline_solve(self._h, _ptr(d), _ptr(u), _ptr(b), _ptr(x)))
        return x

    @property
    def slices(self) -> np.ndarray:
        n = C.c_int32()
        _check(load_library().hines_host_pipeline_slices(self._h, C.byref(n), None, 0))
        out = np.empty(n.value + 1, np.int64)
        _check(load_library().hines_host_pipeline_slices(self._h, C.byref(n), out.ctypes.data, len(out)))
        return out

    def close(self):
        if self._h is not None:
            load_library().hines_host_pipeline_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def partition_cells(cell_offsets, nparts: int):
    """hines_partition_cells: (cell_part int32[ncells], part_cost int64[nparts]) -- longest-processing-time-first deal of
    the cells to nparts devices by their unknowns (no exchange step: cells are independent)."""
    offs = np.ascontiguousarray(cell_offsets, dtype=np.int64)
    part = np.empty(len(offs) - 1, np.int32)
    cost = np.empty(nparts, np.int64)
    _check(load_library().hines_partition_cells(offs.ctypes.data, len(offs) - 1, int(nparts), part.ctypes.data, cost.ctypes.data))
    return part, cost


def reroot(parent, cell_offsets):
    """hines_reroot (f2): per cell the root that minimises the tree's depth and the breadth-first
    renumbering.  Returns a dict: new_parent int32[N] (cell-local), perm int64[N] (new -> old, global), u_src int64[N],
    root / depth_before / depth_after int32[ncells]."""
    par = np.ascontiguousarray(parent, dtype=np.int32)
    offs = np.ascontiguousarray(cell_offsets, dtype=np.int64)
    n, nc = len(par), len(offs) - 1
    out = dict(new_parent=np.empty(n, np.int32), perm=np.empty(n, np.int64), u_src=np.empty(n, np.int64),
               root=np.empty(nc, np.int32), depth_before=np.empty(nc, np.int32), depth_after=np.empty(nc, np.int32))
    _check(load_library().hines_reroot(par.ctypes.data, offs.ctypes.data, nc, out["new_parent"].ctypes.data,
                                       out["perm"].ctypes.data, out["u_src"].ctypes.data, out["root"].ctypes.data,
                                       out["depth_before"].ctypes.data, out["depth_after"].ctypes.data))
    return out


def gather(dst, src, index, dtype=F64, stream=None):
    """hines_gather: dst[k] = src[index[k]] on the device (index: int64 CUDA tensor)."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    _check(load_library().hines_gather(_ptr(dst), _ptr(src), _ptr(index), int(index.numel()), int(dtype), stream))
    return dst


def scatter(dst, src, index, dtype=F64, stream=None):
    """hines_scatter: dst[index[k]] = src[k] on the device."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    _check(load_library().hines_scatter(_ptr(dst), _ptr(src), _ptr(index), int(index.numel()), int(dtype), stream))
    return dst


STATIC_SCRATCH_BYTES = 8388608


def solve_static(parent, cell_offsets, d, u, b, x, dtype=F64, stream=None):
    """hines_solve_static: the entry point that allocates nothing (no plan; scratch in a static __device__ array of
    STATIC_SCRATCH_BYTES inside the library).  parent (int32, cell-local) and cell_offsets (int64) are DEVICE arrays like
    d, u, b, x (torch CUDA tensors or raw addresses); ncells and n come from cell_offsets' / d's lengths."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    ncells, n = int(cell_offsets.numel()) - 1, int(d.numel())
    _check(load_library().hines_solve_static(_ptr(parent), _ptr(cell_offsets), ncells, n, _ptr(d), _ptr(u), _ptr(b), _ptr(x),
                                             int(dtype), stream))
    return x


def version() -> str:
    return load_library().hines_version().decode()
