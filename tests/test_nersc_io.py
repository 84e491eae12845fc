"""Host-side NERSC-format reader / writer against an independent numpy writer / parser
of the same public format written here in the test: bit-exact links in the canonical Eq. (5) order, checksum, link trace,
two-row reconstruction, fp32 files, little-endian files, and the error paths.  CPU only, no CUDA call."""
import os

import numpy as np
import pytest
import torch

from oracle import smear as osmear
from paper_2306_01098_b200 import binding, inputs, layout


def _thin_lex(L, seed):
    s = torch.arange(inputs.volume(L), dtype=torch.int64)
    return inputs.thin_links(L, seed, s, 0.3).numpy()                      # [V(lex), 4, 3, 3]


def _plaquette(L, U):
    G = osmear._grid(L, U)
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            P, _ = osmear.path_product(G, (mu + 1, nu + 1, -(mu + 1), -(nu + 1)))
            tot += np.trace(P, axis1=-2, axis2=-1).real.mean() / 3.0
    return tot / 6.0


def _numpy_write(path, L, U, rows, dtype, plaq, corrupt_checksum=False):
    """Independent writer: file order is lexicographic sites, mu, rows, columns, (re, im)."""
    data = U[:, :, :rows, :]                                               # [V, 4, rows, 3] complex
    flat = np.stack([data.real, data.imag], axis=-1).astype(dtype)         # dtype carries the byte order
    raw = flat.tobytes()
    words = np.frombuffer(raw, dtype=">u4" if dtype.startswith(">") else "<u4")
    checksum = int(words.astype(np.uint64).sum() & 0xFFFFFFFF)
    fp = {">f8": "IEEE64BIG", ">f4": "IEEE32BIG", "<f8": "IEEE64LITTLE", "<f4": "IEEE32LITTLE"}[dtype]
    lt = np.trace(U, axis1=-2, axis2=-1).real.mean() / 3.0
    hdr = ["BEGIN_HEADER", "HDR_VERSION = 1.0", "DATATYPE = " + ("4D_SU3_GAUGE_3x3" if rows == 3 else "4D_SU3_GAUGE")]
    hdr += [f"DIMENSION_{d + 1} = {L[d]}" for d in range(4)]
    hdr += [f"LINK_TRACE = {lt:.12f}", f"PLAQUETTE = {plaq:.12f}", "ENSEMBLE_ID = synthetic",
            f"CHECKSUM = {(checksum ^ 1) if corrupt_checksum else checksum:x}", f"FLOATING_POINT = {fp}", "END_HEADER"]
    with open(path, "wb") as f:
        f.write(("\n".join(hdr) + "\n").encode())
        f.write(raw)
    return checksum, lt


def _canonical(L, U):
    return np.ascontiguousarray(U[layout.lex_of_eo(L).numpy()].transpose(1, 0, 2, 3))      # [4, V(eo), 3, 3]


@pytest.mark.parametrize("rows,dtype", [(3, ">f8"), (2, ">f8"), (3, ">f4"), (2, "<f8"), (3, "<f4")])
def test_read_matches_independent_writer(tmp_path, rows, dtype):
    L = (4, 6, 8, 4)
    U = _thin_lex(L, 31)
    plaq = _plaquette(L, U)
    path = str(tmp_path / "cfg.nersc")
    _, lt = _numpy_write(path, L, U, rows, dtype, plaq)
    info = binding.nersc_info(path)
    assert info["L"] == L and info["rows"] == rows and info["real_bytes"] == int(dtype[2])
    assert abs(info["plaquette"] - plaq) < 1e-11 and abs(info["link_trace"] - lt) < 1e-11
    got = binding.nersc_read(path).numpy()
    ref = _canonical(L, U)
    if dtype.endswith("f4"):
        ref = ref.astype(np.complex64).astype(np.complex128)
    if rows == 3:
        assert np.array_equal(got, ref)                                    # bit-exact, every link in its Eq. (5) slot
    else:
        assert np.array_equal(got[:, :, :2], ref[:, :, :2])
        assert np.abs(got[:, :, 2] - ref[:, :, 2]).max() < 1e-15           # row 2 = conj(row0 x row1)
    # an SU(3) configuration: the plaquette of what was read equals the header's
    assert abs(_plaquette(L, got[:, layout.eo_of_lex(L).numpy()].transpose(1, 0, 2, 3)) - plaq) < 1e-6


def test_library_writer_roundtrip_and_independent_parse(tmp_path):
    L = (4, 4, 6, 8)
    U = _thin_lex(L, 32)
    can = torch.from_numpy(_canonical(L, U))
    plaq = _plaquette(L, U)
    for rows in (3, 2):
        path = str(tmp_path / f"w{rows}.nersc")
        # a header PLAQUETTE that is not the links' own is refused on reading (the value used to be parsed and
        # ignored); 0 means "not known" and is not checked
        binding.nersc_write(path, can, L, rows=rows, plaquette=0.5)
        with pytest.raises(binding.HisqError) as e:
            binding.nersc_read(path)
        assert e.value.code == binding.HISQ_EIO
        binding.nersc_write(path, can, L, rows=rows, plaquette=plaq)
        back = binding.nersc_read(path).numpy()
        assert np.array_equal(back[:, :, :2], can.numpy()[:, :, :2])
        assert np.abs(back - can.numpy()).max() < 1e-15
        # parse the library's file with numpy only
        blob = open(path, "rb").read()
        head, raw = blob.split(b"END_HEADER\n", 1)
        kv = dict(line.split(" = ") for line in head.decode().splitlines() if " = " in line)
        assert kv["FLOATING_POINT"] == "IEEE64BIG" and [int(kv[f"DIMENSION_{d + 1}"]) for d in range(4)] == list(L)
        words = np.frombuffer(raw, dtype=">u4")
        assert int(words.astype(np.uint64).sum() & 0xFFFFFFFF) == int(kv["CHECKSUM"], 16)
        vals = np.frombuffer(raw, dtype=">f8").reshape(-1, 4, rows, 3, 2)
        assert np.array_equal(vals[..., 0] + 1j * vals[..., 1], U[:, :, :rows, :])
        assert abs(float(kv["LINK_TRACE"]) - np.trace(U, axis1=-2, axis2=-1).real.mean() / 3.0) < 1e-11


def test_error_paths(tmp_path):
    L = (4, 4, 4, 4)
    U = _thin_lex(L, 33)
    lib = binding.load_library()
    buf = torch.empty((4, 256, 3, 3), dtype=torch.complex128)
    def read(p, nbytes=buf.numel() * 16):
        return lib.hisq_nersc_read(str(p).encode(), buf.data_ptr(), nbytes)
    good = tmp_path / "good.nersc"
    _numpy_write(str(good), L, U, 3, ">f8", 0.0)
    assert read(good) == 0
    assert read(tmp_path / "missing.nersc") == binding.HISQ_EIO
    assert read(good, 100) == binding.HISQ_EINVAL                           # buffer too small
    bad = tmp_path / "badsum.nersc"
    _numpy_write(str(bad), L, U, 3, ">f8", 0.0, corrupt_checksum=True)
    assert read(bad) == binding.HISQ_EIO
    blob = good.read_bytes()
    flipped = tmp_path / "flipped.nersc"
    flipped.write_bytes(blob[:-9] + bytes([blob[-9] ^ 0x10]) + blob[-8:])   # one bit of one link
    assert read(flipped) == binding.HISQ_EIO
    short = tmp_path / "short.nersc"
    short.write_bytes(blob[:-64])
    assert read(short) == binding.HISQ_EIO
    nohdr = tmp_path / "nohdr.nersc"
    nohdr.write_bytes(b"hello\n" + blob)
    assert read(nohdr) == binding.HISQ_EINVAL
    odd = tmp_path / "odd.nersc"
    Lo = (3, 4, 4, 4)
    _numpy_write(str(odd), Lo, U[:192], 3, ">f8", 0.0)
    assert binding.nersc_info(str(odd))["L"] == Lo and read(odd) == binding.HISQ_EINVAL
    with pytest.raises(binding.HisqError):
        binding.nersc_read(str(tmp_path / "missing.nersc"))
    # a file without CHECKSUM, or one that declares non-periodic links, is refused rather than accepted
    nosum = tmp_path / "nosum.nersc"
    head, raw = blob.split(b"END_HEADER\n", 1)
    nosum.write_bytes(b"\n".join(l for l in head.split(b"\n") if not l.startswith(b"CHECKSUM")) + b"END_HEADER\n" + raw)
    assert read(nosum) == binding.HISQ_EINVAL
    anti = tmp_path / "anti.nersc"
    anti.write_bytes(head + b"BOUNDARY_4 = ANTIPERIODIC\nEND_HEADER\n" + raw)
    assert read(anti) == binding.HISQ_EINVAL
