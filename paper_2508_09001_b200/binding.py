"""Thin ctypes binding of libretro.so (include/retro.h): argument marshalling only.

Every function has the name of its C entry point and takes torch tensors (device memory, owned by the
caller) whose data pointers are passed through; nothing is computed here.  If the library is missing it is
built with nvcc; if that fails the import raises — there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import math
from typing import Optional

import torch

from . import build as _build

RETRO_OK = 0
RETRO_ERR_ARG, RETRO_ERR_UNSUPPORTED, RETRO_ERR_WORKSPACE, RETRO_ERR_CUDA = -1, -2, -3, -4
RETRO_F32, RETRO_BF16 = 0, 1
RETRO_GROUP_SUM, RETRO_GROUP_MAX = 0, 1

EXPORTED = [
    "retro_workspace_bytes", "retro_workspace_init", "retro_error_string", "retro_last_cuda_error",
    "retro_version", "retro_update_page_bounds", "retro_select_pages", "retro_sparse_attend",
    "retro_merge_output_cache", "retro_append_kv", "retro_decode_step", "retro_decode_step_host",
    "retro_window_advance", "retro_window_advance_layers", "retro_update_kv",
    "retro_budget_policy", "retro_build_mask", "retro_step_diagnostics", "retro_decode_step_part",
    "retro_launches_per_step", "retro_decode_steps_host", "retro_debug_status",
]


class RetroDesc(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "batch", "num_q_heads", "num_kv_heads", "head_dim", "page_size", "max_pages_per_seq", "max_sel_pages",
        "num_phys_pages", "window", "dtype", "group_reduce", "force_last_page")] + [("sm_scale", C.c_float),
                                                                                      ("cache_dtype", C.c_int32)]

    @property
    def group(self):
        return self.num_q_heads // self.num_kv_heads

    @property
    def torch_dtype(self):
        return torch.bfloat16 if self.dtype == RETRO_BF16 else torch.float32


class RetroLayerState(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in (
        "k_pages", "v_pages", "block_table", "seq_lens", "budget_pages", "bounds", "last_loaded", "sel_pages",
        "sel_prev", "sel_count", "part_o", "part_lse", "cache_o", "cache_lse", "cache_pos", "workspace")] + [
        ("workspace_bytes", C.c_size_t)]


class RetroStepIO(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("qkv_new", "q_win", "q_pos", "out")]


class RetroError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = _lib().retro_error_string(code).decode()
        extra = f" (cudaError {_lib().retro_last_cuda_error()})" if code == RETRO_ERR_CUDA else ""
        super().__init__(f"{where}: {msg}{extra}")


_LIB = None
_LIB_PATH = None     # None: the release build (paper_2508_09001_b200/lib/libretro.so)


def _lib():
    global _LIB
    if _LIB is None:
        global _LIB_PATH
        path = _LIB_PATH if _LIB_PATH is not None else _build.build()   # no-op when up to date; raises if nvcc fails
        _LIB_PATH = path
        lib = C.CDLL(path)
        lib.retro_error_string.restype = C.c_char_p
        lib.retro_error_string.argtypes = [C.c_int]
        for name in EXPORTED:
            getattr(lib, name)          # fail loudly on a missing symbol
        _LIB = lib
    return _LIB


def library_path() -> str:
    _lib()
    return _LIB_PATH


def use_library(path: Optional[str] = None):
    """Load another build of the library (e.g. build.build_debug(): device-side index validation); None = the
    release build.  Affects every later call of this module."""
    global _LIB, _LIB_PATH
    _LIB, _LIB_PATH = None, path
    _lib()


def retro_debug_status(desc, workspace, stream=None):
    """(enabled, violations, last_code) of a -DRETRO_DEBUG_CHECKS build; (0, 0, 0) in the release build."""
    en, n, code = C.c_int32(0), C.c_uint32(0), C.c_uint32(0)
    _check(_lib().retro_debug_status(C.byref(desc), _p(workspace), C.c_size_t(workspace.numel()), C.byref(en),
                                     C.byref(n), C.byref(code), _stream(stream)), "retro_debug_status")
    return en.value, n.value, code.value


def _p(t: Optional[torch.Tensor]):
    if t is None:
        return C.c_void_p(0)
    assert t.is_contiguous(), "libretro takes contiguous tensors"
    return C.c_void_p(t.data_ptr())


def _stream(stream) -> C.c_void_p:
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _check(rc: int, where: str):
    if rc != RETRO_OK:
        raise RetroError(rc, where)


def make_desc(batch, num_q_heads, num_kv_heads, head_dim, page_size, max_pages_per_seq, max_sel_pages,
              num_phys_pages, window, dtype, group_reduce=RETRO_GROUP_SUM, force_last_page=1,
              sm_scale=None, cache_dtype=RETRO_F32) -> RetroDesc:
    if isinstance(dtype, torch.dtype):
        dtype = RETRO_BF16 if dtype == torch.bfloat16 else RETRO_F32
    elif isinstance(dtype, str):
        dtype = RETRO_BF16 if dtype == "bf16" else RETRO_F32
    return RetroDesc(batch, num_q_heads, num_kv_heads, head_dim, page_size, max_pages_per_seq, max_sel_pages,
                     num_phys_pages, window, dtype, group_reduce, int(force_last_page),
                     1.0 / math.sqrt(head_dim) if sm_scale is None else sm_scale, int(cache_dtype))


def retro_version() -> int:
    return _lib().retro_version()


def retro_error_string(code: int) -> str:
    return _lib().retro_error_string(code).decode()


def retro_last_cuda_error() -> int:
    return _lib().retro_last_cuda_error()


def retro_workspace_bytes(desc: RetroDesc) -> int:
    n = C.c_size_t(0)
    _check(_lib().retro_workspace_bytes(C.byref(desc), C.byref(n)), "retro_workspace_bytes")
    return n.value


def retro_workspace_init(desc, workspace, stream=None):
    _check(_lib().retro_workspace_init(C.byref(desc), _p(workspace), C.c_size_t(workspace.numel()),
                                       _stream(stream)), "retro_workspace_init")


def retro_update_page_bounds(desc, k_pages, block_table, seq_lens, pos_begin, max_touched_pages, bounds, stream=None):
    _check(_lib().retro_update_page_bounds(C.byref(desc), _p(k_pages), _p(block_table), _p(seq_lens), _p(pos_begin),
                                           C.c_int32(max_touched_pages), _p(bounds), _stream(stream)),
           "retro_update_page_bounds")


def retro_select_pages(desc, q_cur, bounds, seq_lens, budget_pages, last_loaded, sel_pages, sel_prev, sel_count,
                       scores_out, workspace, stream=None):
    _check(_lib().retro_select_pages(C.byref(desc), _p(q_cur), _p(bounds), _p(seq_lens), _p(budget_pages),
                                     _p(last_loaded), _p(sel_pages), _p(sel_prev), _p(sel_count), _p(scores_out),
                                     _p(workspace), C.c_size_t(workspace.numel()), _stream(stream)),
           "retro_select_pages")


def retro_sparse_attend(desc, q_win, q_pos, k_pages, v_pages, block_table, seq_lens, sel_pages, sel_prev, sel_count,
                        part_o, part_lse, workspace, stream=None):
    _check(_lib().retro_sparse_attend(C.byref(desc), _p(q_win), _p(q_pos), _p(k_pages), _p(v_pages), _p(block_table),
                                      _p(seq_lens), _p(sel_pages), _p(sel_prev), _p(sel_count), _p(part_o),
                                      _p(part_lse), _p(workspace), C.c_size_t(workspace.numel()), _stream(stream)),
           "retro_sparse_attend")


def retro_merge_output_cache(desc, part_o, part_lse, q_pos, seq_lens, cache_o, cache_lse, cache_pos, out, out_lse,
                             stream=None):
    _check(_lib().retro_merge_output_cache(C.byref(desc), _p(part_o), _p(part_lse), _p(q_pos), _p(seq_lens),
                                           _p(cache_o), _p(cache_lse), _p(cache_pos), _p(out), _p(out_lse),
                                           _stream(stream)), "retro_merge_output_cache")


def retro_append_kv(desc, k_new, v_new, block_table, seq_lens, k_pages, v_pages, stream=None):
    _check(_lib().retro_append_kv(C.byref(desc), _p(k_new), _p(v_new), _p(block_table), _p(seq_lens), _p(k_pages),
                                  _p(v_pages), _stream(stream)), "retro_append_kv")


def retro_window_advance(desc, q_new_or_pool, step_counter, pool_steps, seq_lens, q_win, q_pos, q_cur_out,
                         stream=None):
    _check(_lib().retro_window_advance(C.byref(desc), _p(q_new_or_pool), _p(step_counter), C.c_int32(pool_steps),
                                       _p(seq_lens), _p(q_win), _p(q_pos), _p(q_cur_out), _stream(stream)),
           "retro_window_advance")


def retro_budget_policy(desc, seq_lens, budget_pages, ratio_permille=150, min_tokens=256, stream=None):
    """Relative budget on the device: budget_pages[b] from seq_lens[b]."""
    _check(_lib().retro_budget_policy(C.byref(desc), _p(seq_lens), C.c_int32(ratio_permille), C.c_int32(min_tokens),
                                      _p(budget_pages), _stream(stream)), "retro_budget_policy")


def retro_build_mask(desc, sel_pages, sel_count, seq_lens, last_loaded, sel_prev, stream=None):
    """Alg. 2 alone for an externally chosen page set."""
    _check(_lib().retro_build_mask(C.byref(desc), _p(sel_pages), _p(sel_count), _p(seq_lens), _p(last_loaded),
                                   _p(sel_prev), _stream(stream)), "retro_build_mask")


def retro_step_diagnostics(desc, sel_pages, sel_prev, sel_count, q_pos, seq_lens, part_lse, out_lse, supp_pages,
                           supp_mass, stream=None):
    """Per-step effective-budget / supplementary-attention counters."""
    _check(_lib().retro_step_diagnostics(C.byref(desc), _p(sel_pages), _p(sel_prev), _p(sel_count), _p(q_pos),
                                         _p(seq_lens), _p(part_lse), _p(out_lse), _p(supp_pages), _p(supp_mass),
                                         _stream(stream)), "retro_step_diagnostics")


def retro_update_kv(desc, k_hat, v_hat, positions, block_table, seq_lens, k_pages, v_pages, stream=None):
    """UpdateKV (Alg. 1 line 2): k_hat / v_hat [B][n_upd][h_k][d], positions [B][n_upd] int32 (-1 = skip)."""
    n_upd = int(positions.shape[1])
    _check(_lib().retro_update_kv(C.byref(desc), _p(k_hat), _p(v_hat), _p(positions), C.c_int32(n_upd),
                                  _p(block_table), _p(seq_lens), _p(k_pages), _p(v_pages), _stream(stream)),
           "retro_update_kv")


def retro_window_advance_layers(desc, table, n_layers, pool_steps, stream=None):
    """table: device int64 tensor [n_layers][6] of device pointers (retro_advance_rec_t records)."""
    _check(_lib().retro_window_advance_layers(C.byref(desc), _p(table), C.c_int32(n_layers), C.c_int32(pool_steps),
                                              _stream(stream)), "retro_window_advance_layers")


def retro_decode_step(desc, state: RetroLayerState, q_win, q_pos, q_cur, out, out_lse=None, stream=None):
    _check(_lib().retro_decode_step(C.byref(desc), C.byref(state), _p(q_win), _p(q_pos), _p(q_cur), _p(out),
                                    _p(out_lse), _stream(stream)), "retro_decode_step")


def retro_decode_step_part(desc, state: RetroLayerState, q_win, q_pos, q_cur, out, part, out_lse=None, stream=None):
    """One kernel of retro_decode_step: part 0 = S1 + S2, part 1 = S3 + S4 (measurement helper)."""
    _check(_lib().retro_decode_step_part(C.byref(desc), C.byref(state), _p(q_win), _p(q_pos), _p(q_cur), _p(out),
                                         _p(out_lse), C.c_int32(part), _stream(stream)), "retro_decode_step_part")


def retro_launches_per_step(desc) -> int:
    n = C.c_int32(0)
    _check(_lib().retro_launches_per_step(C.byref(desc), C.byref(n)), "retro_launches_per_step")
    return n.value


def retro_decode_step_host(desc, state: RetroLayerState, io: RetroStepIO, host_qkv_new, host_out, stream=None):
    """host_qkv_new: pinned host tensor holding [q_new | k_new | v_new] back to back."""
    _check(_lib().retro_decode_step_host(C.byref(desc), C.byref(state), C.byref(io), _p(host_qkv_new), _p(host_out),
                                         _stream(stream)), "retro_decode_step_host")


def retro_decode_steps_host(desc, states, ios, host_qkv_new, host_out, stream=None):
    """All layers of one decode step with one copy in and one copy out (states / ios: lists of the C structs; the
    ios' qkv_new / out buffers must be consecutive slices of one device buffer each)."""
    n = len(states)
    st_arr = (RetroLayerState * n)(*states)
    io_arr = (RetroStepIO * n)(*ios)
    _check(_lib().retro_decode_steps_host(C.byref(desc), st_arr, io_arr, C.c_int32(n), _p(host_qkv_new), _p(host_out),
                                          _stream(stream)), "retro_decode_steps_host")


class LayerBuffers:
    """Caller-side allocation of one layer's device buffers (torch only allocates) + the C state struct."""

    def __init__(self, desc: RetroDesc, k_pages, v_pages, block_table, seq_lens, budget_pages, device="cuda"):
        d = desc
        dev = torch.device(device)
        dt = d.torch_dtype
        B, hq, hk, D, w = d.batch, d.num_q_heads, d.num_kv_heads, d.head_dim, d.window
        self.desc = d
        self.k_pages, self.v_pages, self.block_table = k_pages, v_pages, block_table
        self.seq_lens, self.budget_pages = seq_lens, budget_pages
        self.bounds = torch.zeros((B, hk, d.max_pages_per_seq, 2, D), dtype=dt, device=dev)
        self.last_loaded = torch.full((B, hk, d.max_pages_per_seq), -1, dtype=torch.int32, device=dev)
        self.sel_pages = torch.full((B, hk, d.max_sel_pages), -1, dtype=torch.int32, device=dev)
        self.sel_prev = torch.full((B, hk, d.max_sel_pages), -1, dtype=torch.int32, device=dev)
        self.sel_count = torch.zeros((B, hk), dtype=torch.int32, device=dev)
        self.part_o = torch.zeros((B, w + 1, hq, D), dtype=torch.float32, device=dev)
        self.part_lse = torch.full((B, w + 1, hq), -math.inf, dtype=torch.float32, device=dev)
        cache_dt = torch.bfloat16 if d.cache_dtype == RETRO_BF16 else torch.float32
        self.cache_o = torch.zeros((B, max(w, 1), hq, D), dtype=cache_dt, device=dev)
        self.cache_lse = torch.full((B, max(w, 1), hq), -math.inf, dtype=torch.float32, device=dev)
        self.cache_pos = torch.full((B, max(w, 1)), -1, dtype=torch.int32, device=dev)
        self.out = torch.zeros((B, w + 1, hq, D), dtype=dt, device=dev)
        self.out_lse = torch.zeros((B, w + 1, hq), dtype=torch.float32, device=dev)
        self.q_win = torch.zeros((B, w + 1, hq, D), dtype=dt, device=dev)
        self.q_pos = torch.full((B, w + 1), -1, dtype=torch.int32, device=dev)
        self.q_cur = torch.zeros((B, hq, D), dtype=dt, device=dev)
        self.workspace = torch.zeros(retro_workspace_bytes(d), dtype=torch.uint8, device=dev)
        retro_workspace_init(d, self.workspace)
        self.state = RetroLayerState(*[t.data_ptr() for t in (
            self.k_pages, self.v_pages, self.block_table, self.seq_lens, self.budget_pages, self.bounds,
            self.last_loaded, self.sel_pages, self.sel_prev, self.sel_count, self.part_o, self.part_lse,
            self.cache_o, self.cache_lse, self.cache_pos, self.workspace)], self.workspace.numel())

    def rebuild_bounds(self, stream=None):
        zero = torch.zeros(self.desc.batch, dtype=torch.int32, device=self.seq_lens.device)
        retro_update_page_bounds(self.desc, self.k_pages, self.block_table, self.seq_lens, zero,
                                 self.desc.max_pages_per_seq, self.bounds, stream)
