"""CPU-only checks of the product's host side (no compute call needs a GPU):
 - the C-ABI library loads and exports every symbol include/npfem.h declares;
 - the create-time plan (npfem_plan_*, plain C++ fp64) agrees with the oracle's create step;
 - the block-sparse operator is A_sys^-1 up to the documented drop rule, and the increment-form
   algebra the kernel uses reproduces the oracle's iterates when evaluated in fp64;
 - argument errors come back as error codes, and creating a handle without CUDA fails loudly.
"""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

import workloads as W
from oracle import npfem_oracle as O
from paper_2011_04332_b200 import NpfemError, NpfemHandle, NpfemPlan, load_library

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
DT = 0.1


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "npfem.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(npfem_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = _declared_functions()
    assert {"npfem_create", "npfem_step", "npfem_destroy", "npfem_last_error",
            "npfem_cell_stride", "npfem_step_host"} <= set(names)
    lib = load_library()
    for name in names:
        assert hasattr(lib, name), f"{name} declared in include/npfem.h but not exported"
        assert ctypes.cast(getattr(lib, name), ctypes.c_void_p).value


@pytest.fixture(scope="module", params=[("rbc", 2), ("plt", 1), ("rbc", 3)])
def cell(request):
    kind, level = request.param
    rest, tris = W.rest_shape(kind, level)
    mat = W.default_material(rest, tris)
    return rest, tris, mat, NpfemPlan(tris, rest, mat, DT), O.OracleCell(tris, rest, mat, DT)


def test_plan_create_step_matches_the_oracle(cell):
    rest, tris, mat, plan, oc = cell
    n, T = rest.shape[0], tris.shape[0]
    info = plan.info()
    assert (info["n_verts"], info["n_tris"], info["n_hinges"]) == (n, T, 3 * T // 2)
    assert info["rest_volume"] == pytest.approx(oc.rest_volume, rel=1e-13)
    assert np.allclose(plan.query("mass"), oc.masses(), rtol=1e-13)
    assert plan.query("mass").sum() == pytest.approx(mat["cell_mass"], rel=1e-13)
    assert np.allclose(plan.query("tri_area"), oc.areas(), rtol=1e-13)
    # indexing is bit-exact: same hinge enumeration, same stencils
    assert np.array_equal(plan.query("hinge_verts").reshape(-1, 4), oc.hinges())
    assert np.allclose(plan.query("hinge_K").reshape(-1, 4), oc.hinge_rows(), rtol=1e-11, atol=1e-13)
    w, r = oc.hinge_weights()
    wr = plan.query("hinge_wr").reshape(-1, 2)
    assert np.allclose(wr[:, 0], w, rtol=1e-12) and np.allclose(wr[:, 1], r, rtol=1e-10, atol=1e-13)
    A = plan.query("system").reshape(n, n)
    assert np.allclose(A, oc.system_matrix(), rtol=1e-11, atol=1e-12)
    # D_m^-1 against the oracle's G = D_m^-T [[-1,1,0],[-1,0,1]]
    dm = plan.query("tri_dminv").reshape(T, 3)
    G = oc.G()
    assert np.allclose(G[:, 0, 1], dm[:, 0], rtol=1e-12)
    assert np.allclose(G[:, 1, 1], dm[:, 1], rtol=1e-10, atol=1e-13)
    assert np.allclose(G[:, 1, 2], dm[:, 2], rtol=1e-12)


def test_internal_ordering_is_a_permutation_and_stays_internal(cell):
    rest, tris, mat, plan, oc = cell
    perm = plan.query("perm")
    assert sorted(perm.tolist()) == list(range(rest.shape[0]))


def test_operator_is_the_inverse_up_to_the_drop_rule(cell):
    rest, tris, mat, plan, oc = cell
    n = rest.shape[0]
    A = oc.system_matrix()
    Tinv = np.linalg.inv(A)
    op = plan.query("operator").reshape(n, n)
    tol = plan.info()["inv_drop_tol"]
    assert tol == pytest.approx(2.0 ** -24)
    kept = op != 0
    assert np.array_equal(kept, kept.T)                                 # symmetric pattern
    assert np.allclose(op[kept], Tinv[kept], rtol=3e-7, atol=0)         # fp32 rounding of kept entries
    dropped_l1 = np.abs(np.where(kept, 0.0, Tinv)).sum(axis=1)
    assert (dropped_l1 <= tol * np.abs(Tinv).sum(axis=1) * (1 + 1e-9)).all()
    # the operator applied to A_sys is the identity to fp32 accuracy
    assert np.abs(op @ A - np.eye(n)).max() < 5e-6
    dense = NpfemPlan(tris, rest, mat, DT, inv_drop_tol=0.0)
    opd = dense.query("operator").reshape(n, n)
    assert np.allclose(opd, Tinv, rtol=3e-7, atol=1e-12)
    assert dense.info()["n_op_blocks"] == dense.info()["n_vblocks"] ** 2


def test_single_tf32_blocks_stay_below_fp32_rounding_of_the_row_sum(cell):
    """Blocks applied as ONE TF32 product (error < 2^-9 per product of truncated operands) may hold
    at most 2^-15 of any row's l1 mass, so their total error stays below 2^-24 ||row||_1 |r|_max."""
    rest, tris, mat, plan, oc = cell
    n = rest.shape[0]
    info = plan.info()
    op = plan.query("operator").reshape(n, n)
    x1 = plan.query("operator_x1").reshape(n, n)
    assert 0 <= info["n_op_blocks_tf32x1"] < info["n_op_blocks"]
    assert np.array_equal(x1[x1 != 0], op[x1 != 0])                     # a subset of the operator
    assert (np.diag(x1) == 0).all()                                     # never the diagonal blocks
    share = np.abs(x1).sum(axis=1) / np.abs(op).sum(axis=1)
    assert share.max() <= 2.0 ** -15 * (1 + 1e-6)
    if n >= 600:                                                        # RBC-3: the tier is really used
        assert info["n_op_blocks_tf32x1"] > info["n_op_blocks"] // 4


def test_fp16_split_operator_is_fp32_equivalent_and_its_single_product_tier_is_bounded(cell):
    """global_mode 3 stores every kept block as hi = fp16(x 2^k), lo = fp16(x 2^k - hi) with a power-of-
    two row scaling: hi + lo must reproduce the fp32 operator to 2^-23 of the row's largest entry
    (rows sit in [2^13, 2^14), fp16 resolves 2^-24 absolute there).  Blocks applied as ONE product
    of the hi parts (error <= 2^-11 per product: both operands rounded to 11 bits) may hold at most
    2^-13 of any row's l1 mass, so their total error stays below 2^-24 ||row||_1 |r|_max."""
    rest, tris, mat, plan, oc = cell
    n = rest.shape[0]
    info = plan.info()
    op = plan.query("operator").reshape(n, n)
    f16 = plan.query("operator_f16").reshape(n, n)
    x1 = plan.query("operator_f16x1").reshape(n, n)
    rowmax = np.abs(op).max(axis=1, keepdims=True)
    assert np.array_equal(f16 != 0, op != 0) or (np.abs(op[(f16 != 0) != (op != 0)]) <= rowmax.max() * 2.0 ** -37).all()
    full = x1 == 0                                                      # three-product blocks: hi + lo
    assert (np.abs(f16 - op)[full] <= (2.0 ** -23 * rowmax * np.ones_like(op))[full]).all()
    single = x1 != 0                                                    # one-product blocks: hi alone
    assert (np.abs(f16 - op)[single] <= (2.0 ** -11 * np.abs(op) + 2.0 ** -37 * rowmax)[single]).all()
    assert np.array_equal(x1[single], f16[single])
    assert (np.diag(x1) == 0).all()                                     # never the diagonal blocks
    assert 0 <= info["n_op_blocks_f16x1"] < info["n_op_blocks"]
    share = np.abs(np.where(single, op, 0.0)).sum(axis=1) / np.abs(op).sum(axis=1)
    assert share.max() <= 2.0 ** -13 * (1 + 1e-6)
    if n >= 600:                                                        # RBC-3: the tier is really used
        assert info["n_op_blocks_f16x1"] > info["n_op_blocks_tf32x1"]
    # the hi parts are fp16 numbers: the library's rounding agrees with numpy's float16
    k = np.round(np.log2(rowmax / np.abs(f16).max(axis=1, keepdims=True)))  # 0: same scaling both sides
    assert (k == 0).all()
    scale = 2.0 ** (13 - np.floor(np.log2(rowmax)))
    hi_np = (op * scale).astype(np.float32).astype(np.float16).astype(np.float64) / scale
    assert np.array_equal(x1[single], hi_np[single])


def test_operator_streams_hold_every_block_once_in_a_uniform_shape(cell):
    """global_mode 3 consumes per-warp streams of 512-byte slots whose shape is the same for every
    warp (per row slot j: na[j] three-product slots, nb[j] one-product slots).  Reading the streams
    back the way the kernel walks them (slot order, descriptors with their swizzle bits, row table)
    must give exactly the fp16 operator: no block lost, none twice, padding slots all zero."""
    rest, tris, mat, plan, oc = cell
    n = rest.shape[0]
    info = plan.info()
    shape = plan.query("stream_shape")
    warps, slots, na, nb = int(shape[0]), int(shape[1]), shape[2:6], shape[6:10]
    assert warps == info["threads_per_cta"] // 32
    assert slots == int(na.sum() + nb.sum()) and 0 < slots <= 64
    assert 4 * warps >= info["n_vblocks"]                               # at most 4 block rows per warp
    stream = plan.query("operator_stream").reshape(n, n)
    f16 = plan.query("operator_f16").reshape(n, n)
    assert np.array_equal(stream, f16)
    # work of the padded streams against the unpadded pair counts: the padding stays moderate
    x1 = plan.query("operator_f16x1").reshape(n, n)
    perm = plan.query("perm")
    nvb = info["n_vblocks"]
    def blocks(M):
        Mp = np.zeros((nvb * 8, nvb * 8)); Mp[:n, :n] = M[np.ix_(perm, perm)]
        return np.abs(Mp).reshape(nvb, 8, nvb, 8).sum(axis=(1, 3)) > 0
    single = blocks(x1)
    full = blocks(f16) & ~single
    mma_needed = 3 * np.ceil(full.sum(axis=1) / 2).sum() + np.ceil(single.sum(axis=1) / 2).sum()
    mma_issued = warps * (3 * na.sum() + 2 * nb.sum())
    assert mma_needed <= mma_issued <= 1.6 * mma_needed + 12 * warps


def _halves(words):
    """uint32 words -> float64 pairs (low half = lower index), as fp16."""
    w = np.asarray(words, dtype=np.uint32)
    lo = (w & 0xffff).astype(np.uint16).view(np.float16).astype(np.float64)
    hi = (w >> 16).astype(np.uint16).view(np.float16).astype(np.float64)
    return lo, hi


@pytest.mark.parametrize("kind,level", [("rbc", 2), ("plt", 1), ("rbc", 3)])
def test_mode3_data_path_emulated_from_the_raw_streams(kind, level):
    """The global_mode-3 product replayed on the CPU from the RAW arrays the kernel loads (stream
    words, slot descriptors, row table, row scales), with the kernel's right-hand-side layout
    (per source block a hi and a lo plane of 8-byte chunks {col g, col g+8} x vertices (2t, 2t+1),
    chunk index (4 g + t) ^ 4 (kb & 7)) and the PTX fragment conventions of mma.m16n8k16 restated
    here: A a0/a1 = rows g / g+8 at k = 2t, 2t+1, a2/a3 the same at k + 8; B b0 = k 2t, 2t+1 at
    n = g, b1 = k + 8; D rows = right-hand-side columns, columns = output vertices.  The result
    must be T r to fp32 accuracy: this pins the host side of the data path (streams, descriptors,
    swizzle, scales) against those conventions without a GPU."""
    rest, tris = W.rest_shape(kind, level)
    mat = W.default_material(rest, tris)
    plan = NpfemPlan(tris, rest, mat, DT)
    n = rest.shape[0]
    shape = plan.query("stream_shape")
    warps, Q, na, nb = int(shape[0]), int(shape[1]), shape[2:6], shape[6:10]
    val = plan.query("stream_val").view(np.uint32).reshape(warps, Q, 32, 4)
    desc = plan.query("stream_desc").view(np.uint32).reshape(warps, 32, 4)
    rows = plan.query("stream_rows").reshape(4, 32)
    row_scale = plan.query("row_scale")
    perm = plan.query("perm")
    nvb = plan.info()["n_vblocks"]
    NP = nvb * 8
    rng = np.random.Generator(np.random.PCG64(23))
    r = np.zeros((NP, 16), dtype=np.float32)                          # internal vertex order, 15 columns + pad
    r[:n, :15] = (rng.standard_normal((n, 15)) * 10.0 ** rng.uniform(-4, 1, size=(1, 15))).astype(np.float32)
    # split pass: per cell (3 columns) scale to max |r| in [2^13, 2^14), fp16 hi / lo, swizzled layout
    buf = np.zeros(nvb * 512, dtype=np.uint8)
    b16 = buf.view(np.uint16)
    cell_exp = []
    for c in range(5):
        mx = np.abs(r[:, 3 * c:3 * c + 3]).max()
        e = int(np.float32(mx).view(np.uint32) >> 23)                   # biased exponent, as the kernel takes it
        e = min(max(e, 14), 254)
        cell_exp.append(e)
    for v in range(NP):
        kb, k = v >> 3, v & 7
        t, odd = k >> 1, k & 1
        for m in range(16):
            x = np.float32(r[v, m] * np.float32(2.0 ** (140 - cell_exp[m // 3]))) if m < 15 else np.float32(0)
            hi = np.float16(x)
            lo = np.float16(np.float32(x) - np.float32(hi))
            g, up = m & 7, m >> 3
            off = kb * 512 + (((g ^ (kb & 7)) * 4 + t) * 8) + up * 4 + odd * 2
            b16[off // 2] = hi.view(np.uint16)
            b16[(off + 256) // 2] = lo.view(np.uint16)
    b32 = buf.view(np.uint32)

    def afrag(off):                                                      # lane's 8 bytes at byte offset off: (a_even, a_odd)
        return b32[off // 4], b32[off // 4 + 1]

    dd = np.zeros((16, NP))
    for w in range(warps):
        q = 0
        for j in range(4):
            ib = int(rows[j, w])
            D = np.zeros((16, 8))
            for u in range(int(na[j] + nb[j])):
                full = u < na[j]
                for pr in range(1 if full else 2):
                    dw = int(desc[w, q & 31, 2 * ((q >> 5) & 1) + pr])
                    A_hi, A_lo = np.zeros((16, 16)), np.zeros((16, 16))
                    B_hi, B_lo = np.zeros((16, 8)), np.zeros((16, 8))
                    for lane in range(32):
                        g, t = lane >> 2, lane & 3
                        for half, o in enumerate(((dw & 0xffff) ^ (lane * 8), (dw >> 16) ^ (lane * 8))):
                            for plane, A in ((0, A_hi), (256, A_lo)):
                                w0, w1 = afrag(o + plane)
                                (x0, x1), (y0, y1) = _halves(w0), _halves(w1)
                                A[g, 2 * t + 8 * half], A[g, 2 * t + 1 + 8 * half] = x0, x1
                                A[g + 8, 2 * t + 8 * half], A[g + 8, 2 * t + 1 + 8 * half] = y0, y1
                        words = val[w, q, lane]
                        bh = words[0:2] if full else words[2 * pr:2 * pr + 2]
                        for half in range(2):
                            x0, x1 = _halves(bh[half])
                            B_hi[2 * t + 8 * half, g], B_hi[2 * t + 1 + 8 * half, g] = x0, x1
                            if full:
                                x0, x1 = _halves(words[2 + half])
                                B_lo[2 * t + 8 * half, g], B_lo[2 * t + 1 + 8 * half, g] = x0, x1
                    D += A_hi @ B_hi
                    if full:
                        D += A_lo @ B_hi + A_hi @ B_lo
                q += 1
            if ib != 255:
                dd[:, ib * 8:ib * 8 + 8] = D
    got = np.zeros((n, 15))
    for v in range(n):
        for m in range(15):
            got[v, m] = dd[m, v] * row_scale[v] * 2.0 ** (cell_exp[m // 3] - 140)
    op = plan.query("operator").reshape(n, n)[np.ix_(perm, perm)]    # internal order
    want = op @ r[:n, :15].astype(np.float64)
    bound = np.abs(op).sum(axis=1, keepdims=True) * np.abs(r[:n, :15]).reshape(n, 5, 3).max(axis=(0, 2)).repeat(3)[None, :]
    assert (np.abs(got - want) <= 4 * 2.0 ** -24 * bound).all()


def test_global_area_term_is_rejected_by_the_cuda_library():
    """The global-area term (reading A-24) exists in the oracle only: the product must say so
    instead of silently ignoring the weight."""
    rest, tris = W.rest_shape("rbc", 2)
    with pytest.raises(NpfemError) as err:
        NpfemPlan(tris, rest, W.default_material(rest, tris, w_garea=0.5), DT)
    assert "oracle only" in str(err.value)
    NpfemPlan(tris, rest, W.default_material(rest, tris, w_garea=0.0, ga_min=0.9, ga_max=1.1), DT)


def test_info_reports_the_occupancy_limiter():
    """ADVICE (round 1): small meshes are limited by tensor-memory columns (64 per CTA, 512 per SM),
    not by the shared memory the plan sizes; npfem_info says so.  RBC-3 fills one SM's shared memory."""
    rest, tris = W.rest_shape("plt", 1)
    info = NpfemPlan(tris, rest, W.default_material(rest, tris), DT).info()
    assert info["tmem_columns"] == 64 and info["ctas_per_sm"] == 8 and info["ctas_per_sm_limiter"] == 2
    rest, tris = W.rest_shape("rbc", 3)
    info = NpfemPlan(tris, rest, W.default_material(rest, tris), DT).info()
    assert info["tmem_columns"] == 512 and info["ctas_per_sm"] == 1 and info["ctas_per_sm_limiter"] == 1
    damped = NpfemPlan(tris, rest, W.default_material(rest, tris, c_alpha=0.01), DT).info()
    assert damped["tmem_columns"] == 512                                 # 6 groups x 80 columns


def test_global_mode_default_and_fallback():
    """Default = the fp16-split streams (3); a plan whose streams would need more than 64 slots per
    warp (here: the dense operator of RBC-3, 81 blocks in every row) falls back to 3xTF32 blocks (2),
    also when mode 3 is asked for explicitly; modes 1 and 2 are honoured as given."""
    rest, tris = W.rest_shape("rbc", 3)
    mat = W.default_material(rest, tris)
    assert NpfemPlan(tris, rest, mat, DT).info()["global_mode"] == 3
    assert NpfemPlan(tris, rest, mat, DT, global_mode=2).info()["global_mode"] == 2
    assert NpfemPlan(tris, rest, mat, DT, global_mode=1).info()["global_mode"] == 1
    dense = NpfemPlan(tris, rest, mat, DT, inv_drop_tol=0.0)
    assert dense.query("stream_shape")[1] > 64
    assert dense.info()["global_mode"] == 2
    assert NpfemPlan(tris, rest, mat, DT, inv_drop_tol=0.0, global_mode=3).info()["global_mode"] == 2
    with pytest.raises(NpfemError):
        dense.query("operator_stream")


def test_fp16_split_product_emulated_in_numpy_is_fp32_equivalent(cell):
    """The arithmetic of the global_mode-3 product, emulated on the CPU with numpy float16: right-
    hand sides scaled per cell by a power of two to max |r| in [2^13, 2^14), split into hi = fp16(x),
    lo = fp16(x - hi); operator rows scaled likewise; three products hi*hi + hi*lo + lo*hi for the
    full-tier blocks, hi*hi for the single-tier blocks, fp32 accumulation.  Against T r in fp64 the
    error must stay at the level of fp32 rounding of the row sums (a few 2^-24 ||row||_1 |r|_max)."""
    rest, tris, mat, plan, oc = cell
    n = rest.shape[0]
    op = plan.query("operator").reshape(n, n)
    x1 = plan.query("operator_f16x1").reshape(n, n)
    single = x1 != 0
    rowmax = np.abs(op).max(axis=1, keepdims=True)
    tscale = 2.0 ** (13 - np.floor(np.log2(rowmax)))
    ts = (op * tscale).astype(np.float32)
    t_hi = ts.astype(np.float16)
    t_lo = (ts - t_hi.astype(np.float32)).astype(np.float16)
    rng = np.random.Generator(np.random.PCG64(11))
    worst = 0.0
    for trial in range(4):
        r = (rng.standard_normal((n, 3)) * 10.0 ** rng.uniform(-6, 2)).astype(np.float32)
        if trial == 3:
            r[rng.random(n) < 0.5] *= 1e-5                               # wide dynamic range inside one cell
        e = int(np.floor(np.log2(np.abs(r).max())))
        rs = r * np.float32(2.0 ** (13 - e))
        r_hi = rs.astype(np.float16)
        r_lo = (rs - r_hi.astype(np.float32)).astype(np.float16)
        th, tl = t_hi.astype(np.float64), np.where(single, 0.0, t_lo.astype(np.float64))
        rh, rl = r_hi.astype(np.float64), r_lo.astype(np.float64)
        full_mask = (~single).astype(np.float64)
        acc = th @ rh + tl @ rh + (th * full_mask) @ rl                  # products exact in fp64; sums rounded below
        got = acc.astype(np.float32).astype(np.float64) / tscale * 2.0 ** (e - 13)
        want = op @ r.astype(np.float64)
        bound = np.abs(op).sum(axis=1, keepdims=True) * np.abs(r).max()
        worst = max(worst, float((np.abs(got - want) / bound).max()))
    assert worst <= 4 * 2.0 ** -24


def test_elements_pair_all_triangles_of_the_icospheres(cell):
    """The local step works on elements = pairs of triangles across a shared edge (a matching of
    the dual graph); on the icospheres the matching is perfect, so E = T/2 threads do the work."""
    rest, tris, mat, plan, oc = cell
    info = plan.info()
    T = tris.shape[0]
    assert 2 * info["n_diamonds"] + (info["n_elements"] - info["n_diamonds"]) == T
    assert info["n_elements"] == T // 2 and info["n_diamonds"] == T // 2
    assert info["threads_per_cta"] >= max(info["n_elements"], rest.shape[0])


def test_increment_form_with_the_kept_operator_reproduces_oracle_iterates():
    """The algebra of the kernel, d <- d + T (f_int(s + d) - (m/h^2) d), evaluated in fp64 with
    the plan's (dropped, fp32-rounded) operator, against the oracle's absolute-form iterates."""
    rest, tris = W.rest_shape("rbc", 2)
    mat = W.default_material(rest, tris)
    plan, oc = NpfemPlan(tris, rest, mat, DT), O.OracleCell(tris, rest, mat, DT)
    n = rest.shape[0]
    op = plan.query("operator").reshape(n, n)
    m = oc.masses()[:, None]
    rng = np.random.default_rng(5)
    x0 = rest + 50.0
    v0 = rng.standard_normal((n, 3)) * 1e-3
    f = rng.standard_normal((n, 3)) * 1e-3
    _, _, iterates, _ = oc.step_cell(x0, v0, f, 6, trace=True)
    s = x0 + DT * v0 + DT * DT * f / m
    d = np.zeros((n, 3))
    for k in range(6):
        e = oc.fint(s + d)
        d = d + op @ (e - m / DT ** 2 * d)
        err = np.abs((s + d) - iterates[k + 1]).max()
        motion = np.abs(iterates[k + 1] - x0).max()
        assert err <= 2e-6 * motion, (k, err, motion)


def test_argument_errors_are_codes_not_crashes():
    rest, tris = W.rest_shape("rbc", 1)
    mat = W.default_material(rest, tris)
    NpfemPlan(tris, rest, mat, DT)
    bad = dict(mat, c_alpha=-0.1)
    with pytest.raises(NpfemError) as e:
        NpfemPlan(tris, rest, bad, DT)
    assert e.value.code == -1 and "damping" in str(e.value)
    with pytest.raises(NpfemError):
        NpfemPlan(tris, rest, dict(mat, s_min=1.2, s_max=1.0), DT)
    with pytest.raises(NpfemError):
        NpfemPlan(tris, rest, mat, 0.0)
    with pytest.raises(NpfemError):
        NpfemPlan(tris[:-1], rest, mat, DT)                              # open mesh
    flipped = tris.copy()
    flipped[3] = flipped[3][[0, 2, 1]]
    with pytest.raises(NpfemError):
        NpfemPlan(flipped, rest, mat, DT)                                # inconsistent orientation
    with pytest.raises(NpfemError):
        NpfemPlan(tris[:, [0, 2, 1]], rest, mat, DT)                     # inward: V0 < 0
    big_rest, big_tris = W.rest_shape("rbc", 4)
    with pytest.raises(NpfemError) as e:
        NpfemPlan(big_tris, big_rest, W.default_material(big_rest, big_tris), DT)
    assert e.value.code == -4
    with pytest.raises(NpfemError):
        NpfemPlan(tris, rest, mat, DT, cells_per_cta=9)


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful on a box without CUDA")
def test_no_cpu_fallback_create_fails_loudly_without_cuda():
    rest, tris = W.rest_shape("rbc", 1)
    with pytest.raises(NpfemError) as e:
        NpfemHandle(tris, rest, W.default_material(rest, tris), DT)
    assert e.value.code == -3


def test_damped_system_matrix_matches_the_oracle_and_negative_damping_is_rejected():
    """NEXT-2 (reading A-20): A_sys = (1/h^2 + c_alpha/h) M + (1 + c_beta/h) L_el + w_vol I."""
    rest, tris = W.rest_shape("rbc", 2)
    mat = W.default_material(rest, tris, c_alpha=0.4, c_beta=0.03)
    plan = NpfemPlan(tris, rest, mat, DT)
    oc = O.OracleCell(tris, rest, mat, DT)
    n = rest.shape[0]
    A = plan.query("system").reshape(n, n)
    assert np.allclose(A, oc.system_matrix(), rtol=1e-11, atol=1e-12)
    undamped = NpfemPlan(tris, rest, W.default_material(rest, tris), DT).query("system").reshape(n, n)
    assert np.abs(A - undamped).max() > 0.1                            # the damping really is in there
    op = plan.query("operator").reshape(n, n)
    assert np.abs(op @ A - np.eye(n)).max() < 5e-6
    with pytest.raises(NpfemError):
        NpfemPlan(tris, rest, dict(mat, c_beta=-1.0), DT)
