"""Shared by the GPU tests (not a test module)."""
import torch

ROW2_TOL = {torch.complex128: 1e-14, torch.complex64: 1e-6}


def assert_pack_round_trip(fld, precision, U, recon=None):
    """unpack(pack(U)) against the INDEPENDENTLY generated canonical tensor U (on the device, already packed into the
    field of `precision`, same real type as that field): 18-real storage gives U back bit for bit; 12-real storage gives
    rows 0 and 1 back bit for bit and rebuilds row 2 = conj(row 0 x row 1) to rounding.  Called before a test takes what
    the device holds as the oracle's input: a fault shared by pack and unpack (say, beyond 2^32 byte offsets at 64^4)
    would otherwise hand the oracle the same damaged field the device sweeps.  One time slice at a time."""
    recon = fld.recon if recon is None else recon
    got = fld.unpack(precision, U.dtype)
    assert got.shape == U.shape
    for t in range(U.shape[0]):
        if recon == 18:
            assert torch.equal(got[t], U[t]), "18-real round trip differs in time slice %d" % t
        else:
            assert torch.equal(got[t][..., :2, :], U[t][..., :2, :]), "12-real round trip: rows 0-1 differ in time slice %d" % t
            d = float((got[t][..., 2, :] - U[t][..., 2, :]).abs().max())
            assert d < ROW2_TOL[U.dtype], "12-real round trip: rebuilt row 2 off by %.2e in time slice %d" % (d, t)
    del got
