"""The C-ABI library builds, loads and exports every symbol include/submatrix.h declares
(no compute calls: this runs without a GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_header_symbols():
    from paper_2004_10811_b200 import build, binding
    path = build.build()
    L = ctypes.CDLL(path)
    hdr = open(os.path.join(ROOT, "include", "submatrix.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(sm_[a-z_]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    for name in sorted(declared):
        assert hasattr(L, name), f"{name} declared in submatrix.h but not exported"
    assert declared == set(binding.EXPORTS)


def test_struct_sizes_match_header():
    """ctypes mirrors must have the C layout (sizes and a few field offsets checked against a tiny C program)."""
    import subprocess, tempfile
    from paper_2004_10811_b200 import binding as B
    src = ('#include <stdio.h>\n#include <stddef.h>\n#include "submatrix.h"\nint main(){printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n", '
           'sizeof(sm_options_t), sizeof(sm_plan_info_t), sizeof(sm_stats_t), offsetof(sm_options_t, overshoot), '
           'offsetof(sm_options_t, mu_guess), offsetof(sm_options_t, mu_start), offsetof(sm_stats_t, mu_guess), '
           'offsetof(sm_options_t, kT), offsetof(sm_options_t, shard_world), offsetof(sm_plan_info_t, index_alg_bytes), '
           'offsetof(sm_plan_info_t, shard_val_begin), sizeof(sm_peaks_t));return 0;}\n')
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c")
        open(c, "w").write(src)
        exe = os.path.join(d, "s")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe], check=True)
        out = subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()
    assert [int(x) for x in out] == [ctypes.sizeof(B.sm_options_t), ctypes.sizeof(B.sm_plan_info_t),
                                     ctypes.sizeof(B.sm_stats_t), B.sm_options_t.overshoot.offset,
                                     B.sm_options_t.mu_guess.offset, B.sm_options_t.mu_start.offset,
                                     B.sm_stats_t.mu_guess.offset, B.sm_options_t.kT.offset,
                                     B.sm_options_t.shard_world.offset, B.sm_plan_info_t.index_alg_bytes.offset,
                                     B.sm_plan_info_t.shard_val_begin.offset, ctypes.sizeof(B.sm_peaks_t)]


def test_strerror_and_missing_library_is_loud(monkeypatch):
    from paper_2004_10811_b200 import binding as B
    assert "structure" in B.sm_strerror(B.SM_ERR_STRUCTURE)
    assert "warning" in B.sm_strerror(B.SM_WARN_MU_NOT_CONVERGED)
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", "/nonexistent/libsubmatrix_b200.so")
    try:
        B.lib()
    except RuntimeError as e:
        assert "no CPU fallback" in str(e)
    else:
        raise AssertionError("missing library must raise")


def test_plan_validation_is_host_logic():
    """Structure errors (readings A1, A3, A6) are detected on the host before any CUDA call, so the
    validation of sm_plan_create can be exercised without a GPU: every malformed input must come back
    as its documented status with *plan == NULL."""
    import numpy as np
    from paper_2004_10811_b200 import binding as B, workloads as W
    L = B.lib()
    m = W.random_block_pattern(nb=12, density=0.3, max_bs=3, seed=1)

    def status(nb=None, blk_size=None, colptr=None, rowidx=None, ngroups=None, grp_ptr=None, grp_cols=None, opt=None):
        a = [np.ascontiguousarray(x) for x in (
            m.blk_size if blk_size is None else blk_size, m.colptr if colptr is None else colptr,
            m.rowidx if rowidx is None else rowidx, m.grp_ptr if grp_ptr is None else grp_ptr,
            m.grp_cols if grp_cols is None else grp_cols)]
        plan = ctypes.c_void_p(0xdead)
        st = L.sm_plan_create(ctypes.byref(plan), m.nb if nb is None else nb, a[0].ctypes.data, a[1].ctypes.data,
                              a[2].ctypes.data, m.ngroups if ngroups is None else ngroups, a[3].ctypes.data,
                              a[4].ctypes.data, opt, None)
        assert st < 0 and not plan.value  # every case below is an error: *plan is reset to NULL
        return st

    cols = m.block_cols()
    gc = m.grp_cols.copy(); gc[0] = gc[1]
    assert status(grp_cols=gc) == B.SM_ERR_STRUCTURE                      # groups not a partition (A6)
    gp = m.grp_ptr.copy(); gp[-1] -= 1
    assert status(grp_ptr=gp) == B.SM_ERR_STRUCTURE                       # groups do not cover all columns
    k = np.nonzero(m.rowidx != cols)[0][0]                                # drop one off-diagonal block: asymmetric (A1)
    cp = m.colptr.copy(); cp[cols[k] + 1:] -= 1
    assert status(rowidx=np.delete(m.rowidx, k), colptr=cp) == B.SM_ERR_STRUCTURE
    k = np.nonzero(m.rowidx == cols)[0][0]                                # drop a diagonal block (A3)
    cp = m.colptr.copy(); cp[cols[k] + 1:] -= 1
    assert status(rowidx=np.delete(m.rowidx, k), colptr=cp) == B.SM_ERR_STRUCTURE
    c = int(np.argmax(np.diff(m.colptr) >= 2))                            # unsorted rows inside a column
    r = m.rowidx.copy(); p0 = m.colptr[c]; r[[p0, p0 + 1]] = r[[p0 + 1, p0]]
    assert status(rowidx=r) == B.SM_ERR_STRUCTURE
    bs = m.blk_size.copy(); bs[3] = 0
    assert status(blk_size=bs) == B.SM_ERR_INVALID_ARG                    # non-positive block size
    assert status(nb=-1) == B.SM_ERR_INVALID_ARG
    assert L.sm_plan_create(None, m.nb, None, None, None, 0, None, None, None, None) == B.SM_ERR_INVALID_ARG


def test_option_validation_is_host_logic():
    """Bad option values (round-2 options: method, kT, shard_rank / shard_world) are rejected before any CUDA
    call, and sm_partition_groups / sm_plan_set_allreduce validate their arguments -- all without a GPU."""
    import numpy as np
    from paper_2004_10811_b200 import binding as B, workloads as W
    L = B.lib()
    m = W.random_block_pattern(nb=12, density=0.3, max_bs=3, seed=1)
    arrs = [np.ascontiguousarray(x) for x in (m.blk_size, m.colptr, m.rowidx, m.grp_ptr, m.grp_cols)]

    def status(**kw):
        opt = B.default_options(**kw)
        plan = ctypes.c_void_p(0xdead)
        st = L.sm_plan_create(ctypes.byref(plan), m.nb, arrs[0].ctypes.data, arrs[1].ctypes.data, arrs[2].ctypes.data,
                              m.ngroups, arrs[3].ctypes.data, arrs[4].ctypes.data, ctypes.byref(opt), None)
        assert st < 0 and not plan.value
        return st

    assert status(method=2) == B.SM_ERR_INVALID_ARG
    assert status(method=1, kT=-1.0) == B.SM_ERR_INVALID_ARG
    assert status(method=1, precision=2) == B.SM_ERR_INVALID_ARG          # the eigendecomposition path is FP64 only
    assert status(precision=5) == B.SM_ERR_INVALID_ARG                    # 0 FP64, 1 TF32, 2 3xTF32, 3 BF16x2, 4 FP16x2
    assert status(precision=-1) == B.SM_ERR_INVALID_ARG
    assert status(shard_rank=2, shard_world=2) == B.SM_ERR_INVALID_ARG
    assert status(shard_rank=0, shard_world=m.ngroups + 1) == B.SM_ERR_INVALID_ARG
    dims = np.array([3, 4, 5], dtype=np.int32)
    first = np.zeros(5, dtype=np.int32)
    assert L.sm_partition_groups(3, dims.ctypes.data, 4, first.ctypes.data) == B.SM_ERR_INVALID_ARG  # world > ngroups
    assert L.sm_partition_groups(3, dims.ctypes.data, 0, first.ctypes.data) == B.SM_ERR_INVALID_ARG
    assert L.sm_partition_groups(3, dims.ctypes.data, 2, None) == B.SM_ERR_INVALID_ARG
    assert L.sm_plan_set_allreduce(None, ctypes.cast(None, B.ALLREDUCE_FN), None) == B.SM_ERR_INVALID_ARG
    assert L.sm_measure_peaks(None, None) == B.SM_ERR_INVALID_ARG
