"""ctypes wrapper around oracle_mla.c -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It never imports paper_2607_02043_b200.kairos (the CUDA binding); inputs come from
paper_2607_02043_b200.workloads (the shared, arithmetic-free generator module) as numpy arrays.

The shared object is compiled on first use with gcc (`-O3 -fopenmp`, plus the widest x86 vector ISA
/proc/cpuinfo reports, encoded in the file name so a library built on another host is never loaded).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_mla.c")
_LIB: Optional[ctypes.CDLL] = None


def _isa_variant() -> tuple[str, list[str]]:
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    toks = set(flags.split())
    if {"avx512f", "avx512vl", "avx512bw", "avx512dq"} <= toks:
        return "avx512", ["-mavx512f", "-mavx512vl", "-mavx512bw", "-mavx512dq", "-mfma", "-mavx2"]
    if {"avx2", "fma"} <= toks:
        return "avx2", ["-mavx2", "-mfma"]
    return "base", []


def lib_path() -> str:
    return os.path.join(_HERE, f"liboracle_{_isa_variant()[0]}.so")


def build(force: bool = False) -> str:
    """Compile oracle_mla.c -> liboracle_<isa>.so beside the source (idempotent)."""
    path = lib_path()
    if not force and os.path.exists(path) and os.path.getmtime(path) >= os.path.getmtime(_SRC):
        return path
    cmd = ["gcc", "-O3", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-fno-math-errno",
           *_isa_variant()[1], "-o", path, _SRC, "-lm"]
    subprocess.run(cmd, check=True, capture_output=True, text=True)
    return path


def _lib() -> ctypes.CDLL:
    global _LIB
    if _LIB is None:
        lib = ctypes.CDLL(build())
        c = ctypes
        vp = c.c_void_p
        lib.oracle_append.argtypes = [vp, c.c_int64, vp, vp, c.c_int32, vp, c.c_int32, c.c_int32]
        lib.oracle_append.restype = c.c_int
        lib.oracle_gather.argtypes = [vp, vp, c.c_int32, vp]
        lib.oracle_gather.restype = c.c_int
        lib.oracle_attend_rows.argtypes = [vp, vp, c.c_int32, vp, vp, c.c_int32, vp, c.c_float, vp, vp]
        lib.oracle_attend_rows.restype = c.c_int
        lib.oracle_mixed_step.argtypes = [vp, c.c_int32, vp, vp, c.c_int32, vp, c.c_int32, c.c_int32, vp, vp,
                                          c.c_float, vp, vp, vp, vp]
        lib.oracle_mixed_step.restype = c.c_int
        lib.oracle_dense_bruteforce.argtypes = [vp, vp, c.c_int32, vp, c.c_int32, vp, c.c_double, vp, vp]
        lib.oracle_dense_bruteforce.restype = c.c_int
        lib.oracle_num_threads.argtypes = []
        lib.oracle_num_threads.restype = c.c_int
        _LIB = lib
    return _LIB


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _u16(a) -> np.ndarray:
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, a.dtype
    return a


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def num_threads() -> int:
    return int(_lib().oracle_num_threads())


def append(pool: np.ndarray, latent: np.ndarray, k_rope: np.ndarray, page_table: np.ndarray, start_pos: int) -> None:
    """In-place paged append (a1). pool uint16 [num_pages,64,576]."""
    assert pool.dtype == np.uint16 and pool.flags.c_contiguous and pool.flags.writeable
    latent, k_rope, page_table = _u16(latent), _u16(k_rope), _i32(page_table)
    n = latent.shape[0]
    assert latent.shape == (n, 512) and k_rope.shape == (n, 64)
    rc = _lib().oracle_append(_p(pool), pool.shape[0], _p(latent), _p(k_rope), n, _p(page_table),
                              page_table.shape[0], int(start_pos))
    if rc != 0:
        raise ValueError("oracle_append: position beyond page table or bad page id")


def gather(pool: np.ndarray, page_table: np.ndarray, n: int) -> np.ndarray:
    page_table = _i32(page_table)
    out = np.empty((n, 576), dtype=np.uint16)
    _lib().oracle_gather(_p(_u16(pool)), _p(page_table), int(n), _p(out))
    return out


def attend_rows(pool, page_tables, table_stride, seq_index, q, n_keys, sigma, want_lse=True):
    """Generic rows: query token i (all 16 heads) sees positions 0..n_keys[i]-1 of sequence seq_index[i]."""
    pool, q = _u16(pool), _u16(q)
    page_tables, seq_index, n_keys = _i32(page_tables), _i32(seq_index), _i32(n_keys)
    nq = q.shape[0]
    assert q.shape == (nq, 16, 576)
    out = np.empty((nq, 16, 512), dtype=np.float32)
    lse = np.empty((nq, 16), dtype=np.float32) if want_lse else None
    rc = _lib().oracle_attend_rows(_p(pool), _p(page_tables), int(table_stride), _p(seq_index), _p(q), nq,
                                   _p(n_keys), ctypes.c_float(sigma), _p(out), _p(lse))
    if rc != 0:
        raise ValueError("oracle_attend_rows: n_keys < 1")
    return out, lse


def mixed_step(pool, q_dec, dec_page_tables, dec_ctx_lens, chunk_len, prefix_len, q_chunk, chunk_page_table, sigma):
    """The mixed step. Returns (out_dec f32 [B,16,512], out_chunk f32 [C,16,512], lse_dec, lse_chunk)."""
    pool = _u16(pool)
    dec_ctx_lens = _i32(dec_ctx_lens)
    B = dec_ctx_lens.shape[0]
    C = int(chunk_len)
    dec_page_tables = _i32(dec_page_tables).reshape(B, -1) if B else np.zeros((0, 1), np.int32)
    q_dec = _u16(q_dec).reshape(B, 16, 576)
    q_chunk = _u16(q_chunk).reshape(C, 16, 576)
    chunk_page_table = _i32(chunk_page_table)
    out_dec = np.empty((B, 16, 512), np.float32)
    out_chunk = np.empty((C, 16, 512), np.float32)
    lse_dec = np.empty((B, 16), np.float32)
    lse_chunk = np.empty((C, 16), np.float32)
    rc = _lib().oracle_mixed_step(_p(pool), B, _p(q_dec), _p(dec_page_tables), dec_page_tables.shape[1],
                                  _p(dec_ctx_lens), C, int(prefix_len), _p(q_chunk), _p(chunk_page_table),
                                  ctypes.c_float(sigma), _p(out_dec), _p(out_chunk), _p(lse_dec), _p(lse_chunk))
    if rc != 0:
        raise ValueError("oracle_mixed_step failed (ctx_len < 1?)")
    return out_dec, out_chunk, lse_dec, lse_chunk


def dense_bruteforce(pool, page_table, n_total, q, n_keys, sigma):
    """Double-precision dense masked softmax attention on one sequence. Returns (out f64, probs f64)."""
    pool, q = _u16(pool), _u16(q)
    page_table, n_keys = _i32(page_table), _i32(n_keys)
    nq = q.shape[0]
    out = np.empty((nq, 16, 512), np.float64)
    probs = np.empty((nq, 16, int(n_total)), np.float64)
    _lib().oracle_dense_bruteforce(_p(pool), _p(page_table), int(n_total), _p(q), nq, _p(n_keys),
                                   ctypes.c_double(sigma), _p(out), _p(probs))
    return out, probs
