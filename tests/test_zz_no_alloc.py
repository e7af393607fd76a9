"""opo_spectrum_noalloc: the spectrum read-out for callers that cannot let the library allocate device memory.

Some users of libopo run it inside a process where a memory pool (PyTorch's caching allocator, an RMM pool, an
instrument-control program's own arena) already holds all of HBM, so a cudaMalloc issued by the library would fail; others
look at the spectrum inside a feedback loop and cannot take the device-wide stall cudaMalloc / cudaFree cause.  For them
include/opo.h offers one call that needs no handle: the tables the transform kernel reads sit in a fixed 192 KiB array that
is part of libopo.so itself, which caps a row at 2^14 points (complex64) or 2^13 (complex128).

What is checked here: the call returns what the existing path -- a handle plus opo_get_fields(.., OPO_DOMAIN_FREQ, ..) --
returns for the same rows, to the tolerance the read-out test of test_gpu_parity.py uses against the oracle (2e-6 / 1e-13),
and, because both run the same kernel on the same table values, bit for bit.  Two calls in a row are made on purpose: the
array is shared by every call and keeps what the previous call left in it, so the second call (same size: tables reused;
other size: tables rewritten) is where a stale or half-written table would show.

This file is named so that pytest collects it last: with `-x` a failure here cannot hide another test.  It makes its own
inputs and does not depend on anything an earlier test did, so it passes alone in a fresh process as well.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"c64": 2e-6, "c128": 1e-13}      # the figures of test_frequency_readout_matches_oracle_fft


def _gpu():
    import torch
    import paper_2410_02532_b200 as P
    return torch, P


def _rows(torch, seed, batch, n, dtype):
    """Seeded complex rows with a coloured spectrum (not white noise: a wrong bin order would show)."""
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((batch, n)) + 1j * rng.standard_normal((batch, n))
    x *= 1.0 + 0.5 * np.cos(2 * np.pi * 3 * np.arange(n) / n)[None, :]
    return torch.from_numpy(x).to(dtype).cuda().contiguous()


def _existing_path(P, log2_n, precision, rows):
    """Spectrum of `rows` through a handle: opo_set_field + opo_get_fields(FREQ).  The physics parameters are
    irrelevant to the read-out; they only have to pass opo_create's validation."""
    o = P.Opo(n_fields=2, log2_n=log2_n, window_s=1e-11, nz_per_pass=2, length_m=1e-3, dk_per_m=0.0, d_eff_m_per_V=14e-12,
              lambda_m=[532e-9, 1064e-9], n_index=[2.23, 2.16], beta1_s_per_m=[0.0, 0.0], beta2_s2_per_m=[0.0, 0.0],
              resonant=[0, 1], R=[0.0, 0.9], precision=precision, batch=rows.shape[0])
    o.set_field(1, rows)
    out = o.get_fields(1, P.WHICH_CURRENT, P.DOMAIN_FREQ)
    o.sync()
    o.close()
    return out


def _rel_l2(a, b):
    a = a.cpu().numpy().astype(np.complex128)
    b = b.cpu().numpy().astype(np.complex128)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def _noalloc(torch, P, rows, out, log2_n, precision):
    P.opo_spectrum_noalloc(rows.data_ptr(), out.data_ptr(), log2_n, rows.shape[0],
                           P.PRECISION_C128 if precision == "c128" else P.PRECISION_C64, torch.cuda.current_stream().cuda_stream)


@pytest.mark.parametrize("precision,log2_n,batch", [("c64", 14, 5), ("c64", 9, 3), ("c128", 13, 2), ("c64", 4, 7)])
def test_two_calls_in_a_row_match_the_handle_path(precision, log2_n, batch):
    torch, P = _gpu()
    dtype = torch.complex128 if precision == "c128" else torch.complex64
    n = 1 << log2_n
    first, second = _rows(torch, 11, batch, n, dtype), _rows(torch, 12, batch, n, dtype)
    want_first, want_second = _existing_path(P, log2_n, precision, first), _existing_path(P, log2_n, precision, second)
    got_first, got_second = torch.empty_like(first), torch.empty_like(second)
    _noalloc(torch, P, first, got_first, log2_n, precision)        # (may be the set-up call of this device)
    _noalloc(torch, P, second, got_second, log2_n, precision)      # finds the tables the first call left behind
    torch.cuda.synchronize()
    for got, want in ((got_first, want_first), (got_second, want_second)):
        assert _rel_l2(got, want) <= TOL[precision]
        assert torch.equal(got, want)                              # same kernel, same table values


def test_changing_the_size_between_calls_rewrites_the_shared_tables():
    """Sizes A, B, A on one stream: each call must see its own tables although all three use the same array."""
    torch, P = _gpu()
    cases = [("c64", 12), ("c128", 10), ("c64", 12), ("c64", 14)]
    rows = [_rows(torch, 20 + i, 2, 1 << l, torch.complex128 if p == "c128" else torch.complex64) for i, (p, l) in enumerate(cases)]
    want = [_existing_path(P, l, p, r) for (p, l), r in zip(cases, rows)]
    got = [torch.empty_like(r) for r in rows]
    for (p, l), r, g in zip(cases, rows, got):
        _noalloc(torch, P, r, g, l, p)
    torch.cuda.synchronize()
    for (p, l), g, w in zip(cases, got, want):
        assert _rel_l2(g, w) <= TOL[p], (p, l)
        assert torch.equal(g, w), (p, l)


def test_in_place_and_no_growth_of_device_memory():
    """dev_out may be dev_in; and once a size has been set up, a call leaves the device's free memory where it was."""
    torch, P = _gpu()
    rows = _rows(torch, 31, 4, 1 << 13, torch.complex64)
    want = _existing_path(P, 13, "c64", rows)
    work = rows.clone()
    _noalloc(torch, P, work, work, 13, "c64")                     # set-up / table upload for this size happens here
    torch.cuda.synchronize()
    assert torch.equal(work, want)
    work.copy_(rows)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    _noalloc(torch, P, work, work, 13, "c64")
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, (free_before, free_after)
    assert torch.equal(work, want)


def test_rows_beyond_the_built_in_table_space_are_refused_with_a_clear_message():
    torch, P = _gpu()
    x = torch.zeros(1 << 15, dtype=torch.complex64, device="cuda")
    for precision, log2_n in ((P.PRECISION_C64, 15), (P.PRECISION_C128, 14)):
        with pytest.raises(P.OpoError) as e:
            P.opo_spectrum_noalloc(x.data_ptr(), x.data_ptr(), log2_n, 1, precision, 0)
        assert e.value.status == P.ERR_UNSUPPORTED
        assert "limit 2^" in str(e.value)
    with pytest.raises(P.OpoError) as e:
        P.opo_spectrum_noalloc(x.data_ptr(), x.data_ptr(), 10, 0, P.PRECISION_C64, 0)
    assert e.value.status == P.ERR_INVALID_ARG
