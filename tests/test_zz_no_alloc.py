"""pp_zsolve_static: the z solve for callers that cannot allocate device memory.

Some users of this library run where cudaMalloc is not an option: inside an application that reserved the whole GPU
for its own pool and forbids the runtime allocator afterwards, as a plug-in that is only handed buffers, or in a loop
that cannot take the device-wide synchronisation an allocation implies.  They cannot build a pp_plan (pp_plan_create
allocates its tables), so the library gives them one plan-free call whose only scratch -- the work line of the singular
(0, 0) system -- is a fixed array inside the library, PP_STATIC_MAX_NZ = 4096 doubles long.

The GPU test runs the call twice in a row on one stream (second call: a shorter line, so it meets what the first call
left in the work line) and compares both results with the plan path's z solve (pp_slab_zsolve on a one-rank slab
plan, i.e. the plan's own z kernels) within the tolerance of the other parity tests.  The shift tables are inputs of
the call, so the test writes them out from Table 2 itself.

This file is named so that pytest collects it last: the suite runs with -x, and a failure here must not hide the
parity tests.  It does not depend on anything the other tests did (it passes alone in a fresh process too).
"""
import numpy as np
import pytest

from gpu_util import TOL, rel_err

P, N, D = 0, 1, 2


def shift_table(bc, n, factor, packed_x):
    """factor * lambda(k(p)) for every stored position p (Table 2; k(p) as the header of pp_zsolve_static says)."""
    ld = np.longdouble
    out = np.empty(n, dtype=np.float64)
    for p in range(n):
        k = p
        if bc == P and packed_x:
            k = 0 if p == 0 else (n // 2 if p == 1 else p // 2)
        if bc == P:
            arg = 2 * ld(np.pi) * k / n
        elif bc == N:
            arg = ld(np.pi) * k / n
        else:
            arg = ld(np.pi) * (k + 1) / n
        out[p] = float(ld(factor) * (-4 * np.sin(arg / 2) ** 2))
    return out


def test_argument_checks_need_no_device():
    import paper_1909_05423_b200.binding as b
    ok = dict(w_ptr=256, nx=8, ny=8, nz=16, bc_z=N, zero_mode=0, scale=1.0, sx_ptr=512, sy_ptr=1024)
    assert b.pp_zsolve_static(**{**ok, "nz": b.PP_STATIC_MAX_NZ + 1}) == b.PP_ERR_STATIC_LIMIT
    assert "4096" in b.strerror(b.PP_ERR_STATIC_LIMIT) and "pp_zsolve_static" in b.strerror(b.PP_ERR_STATIC_LIMIT)
    assert b.pp_zsolve_static(**{**ok, "w_ptr": 0}) == 5
    assert b.pp_zsolve_static(**{**ok, "sx_ptr": 0}) == 5
    assert b.pp_zsolve_static(**{**ok, "bc_z": P}) == 1            # periodic z is not offered here
    assert b.pp_zsolve_static(**{**ok, "bc_z": D, "zero_mode": 1}) == 1
    assert b.pp_zsolve_static(**{**ok, "zero_mode": 3}) == 1
    assert b.pp_zsolve_static(**{**ok, "nz": 1}) == 1
    assert b.pp_zsolve_static(**{**ok, "scale": float("nan")}) == 1
    assert b.pp_zsolve_static(**{**ok, "w_ptr": 260}) == 1         # not 8-byte aligned


# (nx, ny, nz, bc, h): first a singular case on a line the plan solves with its partitioned kernel, then a
# shorter singular one of odd length (same kernel on both sides), a packed periodic-x table, a Dirichlet z, the limit
CASES = [
    [(64, 32, 256, (N, N, N), (0.11, 0.07, 0.13)), (32, 16, 37, (N, N, N), (0.2, 0.3, 0.25))],
    [(32, 64, 100, (P, P, N), (0.05, 0.05, 0.05)), (64, 16, 96, (P, N, D), (0.1, 0.2, 0.15))],
    [(16, 8, 4096, (N, P, N), (0.3, 0.3, 0.1)), (8, 16, 4095, (D, N, D), (0.3, 0.3, 0.2))],
]


@pytest.mark.gpu
@pytest.mark.parametrize("pair", CASES)
def test_two_calls_in_a_row_match_the_plan_path(pair):
    import torch
    import paper_1909_05423_b200.binding as b
    stream = torch.cuda.current_stream().cuda_stream
    runs = []
    for seed, (nx, ny, nz, bc, h) in enumerate(pair):
        rng = np.random.default_rng(1909 + seed)
        w0 = rng.standard_normal((nz, ny, nx))
        dz2 = np.longdouble(h[2]) ** 2
        sx = torch.from_numpy(shift_table(bc[0], nx, dz2 / np.longdouble(h[0]) ** 2, True)).cuda()
        sy = torch.from_numpy(shift_table(bc[1], ny, dz2 / np.longdouble(h[1]) ** 2, False)).cuda()
        singular = all(c != D for c in bc)
        scale = float(dz2 / (np.longdouble(nx) * ny))
        w = torch.from_numpy(w0).cuda()
        ref = torch.from_numpy(w0).cuda()
        st, sp = b.pp_slab_plan_create(1, 0, nx, ny, nz, h[0], h[1], h[2], *bc)
        assert st == 0, b.strerror(st)
        runs.append((w, ref, sx, sy, sp, nx, ny, nz, bc, singular, scale))
    # the two static calls back to back, nothing in between
    for w, ref, sx, sy, sp, nx, ny, nz, bc, singular, scale in runs:
        st = b.pp_zsolve_static(w.data_ptr(), nx, ny, nz, bc[2], 1 if singular else 0, scale, sx.data_ptr(), sy.data_ptr(), stream)
        assert st == 0, b.strerror(st)
    for w, ref, sx, sy, sp, nx, ny, nz, bc, singular, scale in runs:
        st = b.pp_slab_zsolve(sp, ref.data_ptr(), stream)
        assert st == 0, b.strerror(st)
    torch.cuda.synchronize()
    for w, ref, sx, sy, sp, nx, ny, nz, bc, singular, scale in runs:
        got, want = w.cpu().numpy(), ref.cpu().numpy()
        assert np.isfinite(got).all()
        assert rel_err(got, want) <= TOL, (nx, ny, nz, bc)
        if singular:    # the line that went through the built-in work line, on its own scale
            assert rel_err(got[:, 0, 0], want[:, 0, 0]) <= TOL, (nx, ny, nz, bc)
        b.pp_slab_plan_destroy(sp)


@pytest.mark.gpu
def test_plane0_convention_and_repeatability():
    """zero_mode = PIN_PLANE0 differs from ZERO_MEAN by a constant on the (0, 0) line only; a repeated call on the same
    input gives the same bits (the work line carries nothing over)."""
    import torch
    import paper_1909_05423_b200.binding as b
    nx, ny, nz, h = 16, 16, 50, (0.1, 0.1, 0.1)
    rng = np.random.default_rng(7)
    w0 = rng.standard_normal((nz, ny, nx))
    sx = torch.from_numpy(shift_table(N, nx, 1.0, True)).cuda()
    sy = torch.from_numpy(shift_table(N, ny, 1.0, False)).cuda()
    out = []
    for mode in (1, 2, 1):
        w = torch.from_numpy(w0).cuda()
        assert b.pp_zsolve_static(w.data_ptr(), nx, ny, nz, N, mode, 0.01, sx.data_ptr(), sy.data_ptr(),
                                  torch.cuda.current_stream().cuda_stream) == 0
        torch.cuda.synchronize()
        out.append(w.cpu().numpy())
    assert np.array_equal(out[0], out[2])
    diff = out[1] - out[0]
    assert np.abs(out[1][0, 0, 0]) == 0.0
    assert np.allclose(diff[:, 0, 0], diff[0, 0, 0], rtol=0, atol=1e-13 * np.abs(out[0]).max())
    diff[:, 0, 0] = 0.0
    assert not diff.any()
    assert abs(out[0][:, 0, 0].mean()) <= 1e-13 * np.abs(out[0]).max()
