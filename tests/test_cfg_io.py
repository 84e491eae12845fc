"""Host-side readers / writers of the ILDG, MILC v5 and openQCD configuration formats
against independent numpy writers / parsers of the same public format descriptions written here in the test (struct,
zlib.crc32, numpy bit operations): bit-exact links in the canonical Eq. (5) order, each format's integrity check, both
byte orders where the format has them, and the error paths.  CPU only, no CUDA call.  No archive file exists in this
container: what is pinned is that reader and writer agree with a second implementation of the stated layout."""
import struct
import zlib

import numpy as np
import pytest
import torch

from paper_2306_01098_b200 import binding, inputs, layout

L = (4, 6, 8, 4)   # Lx, Ly, Lz, Lt: all different enough to catch a swapped axis


def _thin_lex(L, seed):
    s = torch.arange(inputs.volume(L), dtype=torch.int64)
    return inputs.thin_links(L, seed, s, 0.3).numpy()                      # [V(lex), 4, 3, 3]


def _canonical(L, U):
    return np.ascontiguousarray(U[layout.lex_of_eo(L).numpy()].transpose(1, 0, 2, 3))      # [4, V(eo), 3, 3]


def _rotl(w, r):
    w = w.astype(np.uint64)
    return (((w << r) | (w >> (32 - r))) & 0xFFFFFFFF).astype(np.uint64)


def _xor(a):
    return int(np.bitwise_xor.reduce(a.astype(np.uint64)))


# ---- ILDG -------------------------------------------------------------------------------------------------------------
def _lime_record(rtype, payload, begin=False, end=False):
    hdr = struct.pack(">IHHQ", 0x456789AB, 1, (0x8000 if begin else 0) | (0x4000 if end else 0), len(payload))
    hdr += rtype.encode().ljust(128, b"\0")
    return hdr + payload + b"\0" * ((8 - len(payload) % 8) % 8)


def _ildg_bytes(L, U, prec, with_checksum=True, corrupt=False):
    flat = np.stack([U.real, U.imag], axis=-1).astype(">f8" if prec == 64 else ">f4")   # [V, 4, 3, 3, 2], x fastest sites
    raw = bytearray(flat.tobytes())
    site = len(raw) // U.shape[0]
    crcs = np.array([zlib.crc32(bytes(raw[s * site:(s + 1) * site])) for s in range(U.shape[0])], dtype=np.uint64)
    ranks = np.arange(U.shape[0], dtype=np.uint64)
    suma, sumb = _xor(_rotl(crcs, ranks % 29)), _xor(_rotl(crcs, ranks % 31))
    if corrupt:
        raw[len(raw) // 2] ^= 0x10
    fmt = (f"<?xml version=\"1.0\"?><ildgFormat><version>1.0</version><field>su3gauge</field><precision>{prec}</precision>"
           f"<lx>{L[0]}</lx><ly>{L[1]}</ly><lz>{L[2]}</lz><lt>{L[3]}</lt></ildgFormat>").encode()
    out = _lime_record("xlf-info", b"synthetic configuration", begin=True) + _lime_record("ildg-format", fmt)
    out += _lime_record("ildg-binary-data", bytes(raw))
    if with_checksum:
        cs = f"<scidacChecksum><version>1.0</version><suma>{suma:08x}</suma><sumb>{sumb:08x}</sumb></scidacChecksum>".encode()
        out += _lime_record("scidac-checksum", cs, end=True)
    return out


@pytest.mark.parametrize("prec", [64, 32])
def test_ildg_read_matches_independent_writer(tmp_path, prec):
    U = _thin_lex(L, 41)
    path = str(tmp_path / "cfg.ildg")
    open(path, "wb").write(_ildg_bytes(L, U, prec))
    info = binding.cfg_info(path, "ildg")
    assert info == {"L": L, "real_bytes": prec // 8}
    got = binding.cfg_read(path, "ildg").numpy()
    want = _canonical(L, U if prec == 64 else U.astype(np.complex64).astype(np.complex128))
    assert np.array_equal(got, want)


def test_ildg_checksum_and_errors(tmp_path):
    U = _thin_lex(L, 42)
    path = str(tmp_path / "cfg.ildg")
    open(path, "wb").write(_ildg_bytes(L, U, 64, with_checksum=False))            # no checksum record: accepted
    assert np.array_equal(binding.cfg_read(path, "ildg").numpy(), _canonical(L, U))
    open(path, "wb").write(_ildg_bytes(L, U, 64, corrupt=True))                   # one flipped bit: the SciDAC sums catch it
    with pytest.raises(binding.HisqError) as e:
        binding.cfg_read(path, "ildg")
    assert e.value.code == binding.HISQ_EIO
    good = _ildg_bytes(L, U, 64)
    open(path, "wb").write(good[:len(good) // 2])                                 # truncated
    with pytest.raises(binding.HisqError):
        binding.cfg_read(path, "ildg")
    open(path, "wb").write(b"\0" * 200)                                           # not a LIME file
    with pytest.raises(binding.HisqError) as e:
        binding.cfg_info(path, "ildg")
    assert e.value.code == binding.HISQ_EINVAL


def _lime_parse(blob):
    recs, o = {}, 0
    while o < len(blob):
        magic, ver, flags, n = struct.unpack(">IHHQ", blob[o:o + 16])
        assert magic == 0x456789AB and ver == 1
        rtype = blob[o + 16:o + 144].split(b"\0")[0].decode()
        recs[rtype] = blob[o + 144:o + 144 + n]
        o += 144 + (n + 7) // 8 * 8
    return recs


@pytest.mark.parametrize("prec", [64, 32])
def test_ildg_write_parsed_by_independent_reader(tmp_path, prec):
    U = _thin_lex(L, 43)
    path = str(tmp_path / "out.ildg")
    binding.cfg_write(path, "ildg", torch.from_numpy(_canonical(L, U)), L, real_bytes=prec // 8)
    recs = _lime_parse(open(path, "rb").read())
    assert f"<precision>{prec}</precision>" in recs["ildg-format"].decode() and f"<lt>{L[3]}</lt>" in recs["ildg-format"].decode()
    flat = np.frombuffer(recs["ildg-binary-data"], dtype=">f8" if prec == 64 else ">f4").reshape(-1, 4, 3, 3, 2)
    back = flat[..., 0] + 1j * flat[..., 1]
    want = U if prec == 64 else U.astype(np.complex64)
    assert np.array_equal(back.astype(np.complex128), want.astype(np.complex128))
    assert np.array_equal(binding.cfg_read(path, "ildg").numpy(), _canonical(L, want.astype(np.complex128)))   # incl. its own checksum


# ---- MILC v5 ----------------------------------------------------------------------------------------------------------
def _milc_bytes(L, U, order="<", corrupt=False, site_list=False):
    flat = np.stack([U.real, U.imag], axis=-1).astype(order + "f4")             # [V, 4, 3, 3, 2]
    raw = bytearray(flat.tobytes())
    words = np.frombuffer(bytes(raw), dtype=order + "u4").astype(np.uint64)
    k = np.arange(words.size, dtype=np.uint64)
    s29, s31 = _xor(_rotl(words, k % 29)), _xor(_rotl(words, k % 31))
    if corrupt:
        raw[1000] ^= 0x01
    hdr = struct.pack(order + "i4i", 20103, *L) + b"Thu Jan  1 00:00:00 1970".ljust(64, b"\0")
    hdr += struct.pack(order + "iII", 1 if site_list else 0, s29, s31)
    assert len(hdr) == 96
    return hdr + bytes(raw)


@pytest.mark.parametrize("order", ["<", ">"])
def test_milc_read_matches_independent_writer(tmp_path, order):
    U = _thin_lex(L, 44)
    path = str(tmp_path / "cfg.milc")
    open(path, "wb").write(_milc_bytes(L, U, order))
    assert binding.cfg_info(path, "milc") == {"L": L, "real_bytes": 4}
    got = binding.cfg_read(path, "milc").numpy()
    assert np.array_equal(got, _canonical(L, U.astype(np.complex64).astype(np.complex128)))


def test_milc_checksum_and_errors(tmp_path):
    U = _thin_lex(L, 45)
    path = str(tmp_path / "cfg.milc")
    open(path, "wb").write(_milc_bytes(L, U, corrupt=True))
    with pytest.raises(binding.HisqError) as e:
        binding.cfg_read(path, "milc")
    assert e.value.code == binding.HISQ_EIO
    open(path, "wb").write(_milc_bytes(L, U, site_list=True))                     # order != 0 is refused, not misread
    with pytest.raises(binding.HisqError) as e:
        binding.cfg_read(path, "milc")
    assert e.value.code == binding.HISQ_EINVAL
    good = _milc_bytes(L, U)
    open(path, "wb").write(good[:-100])
    with pytest.raises(binding.HisqError):
        binding.cfg_read(path, "milc")
    open(path, "wb").write(struct.pack("<i", 12345) + good[4:])                   # wrong magic number
    with pytest.raises(binding.HisqError) as e:
        binding.cfg_info(path, "milc")
    assert e.value.code == binding.HISQ_EINVAL


def test_milc_write_parsed_by_independent_reader(tmp_path):
    U = _thin_lex(L, 46)
    path = str(tmp_path / "out.milc")
    binding.cfg_write(path, "milc", torch.from_numpy(_canonical(L, U)), L, real_bytes=4)
    blob = open(path, "rb").read()
    assert blob == _milc_bytes(L, U)[:20] + blob[20:84] + _milc_bytes(L, U)[84:]   # everything but the time stamp, bit for bit


# ---- openQCD -----------------------------------------------------------------------------------------------------------
def _plaquette3(L, U):
    """Average of Re tr over all plaquettes (3 for unit links), by np.roll on the [t, z, y, x] grid."""
    G = U.reshape(L[3], L[2], L[1], L[0], 4, 3, 3)
    ax = {0: 3, 1: 2, 2: 1, 3: 0}
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            a, b = G[..., mu, :, :], np.roll(G[..., nu, :, :], -1, axis=ax[mu])
            c, d = np.roll(G[..., mu, :, :], -1, axis=ax[nu]), G[..., nu, :, :]
            P = a @ b @ np.conj(np.swapaxes(c, -1, -2)) @ np.conj(np.swapaxes(d, -1, -2))
            tot += np.trace(P, axis1=-2, axis2=-1).real.mean()
    return tot / 6.0


def _openqcd_bytes(L, U, plaq=None):
    G = U.reshape(L[3], L[2], L[1], L[0], 4, 3, 3)                               # [t, z, y, x, mu]
    out = bytearray(struct.pack("<4id", L[3], L[0], L[1], L[2], _plaquette3(L, U) if plaq is None else plaq))
    ours = {0: 3, 1: 0, 2: 1, 3: 2}                                               # openQCD direction -> our mu
    for t in range(L[3]):
        for x in range(L[0]):
            for y in range(L[1]):
                for z in range(L[2]):
                    if (t + x + y + z) % 2 == 0:
                        continue
                    for mo in range(4):
                        mu = ours[mo]
                        c = [x, y, z, t]
                        fw = G[t, z, y, x, mu]
                        c[mu] = (c[mu] - 1) % L[mu]
                        bw = G[c[3], c[2], c[1], c[0], mu]
                        for m in (fw, bw):
                            out += np.stack([m.real, m.imag], axis=-1).astype("<f8").tobytes()
    return bytes(out)


def test_openqcd_read_matches_independent_writer(tmp_path):
    U = _thin_lex(L, 47)
    path = str(tmp_path / "cfg.oqcd")
    open(path, "wb").write(_openqcd_bytes(L, U))
    assert binding.cfg_info(path, "openqcd") == {"L": L, "real_bytes": 8}
    assert np.array_equal(binding.cfg_read(path, "openqcd").numpy(), _canonical(L, U))


def test_openqcd_plaquette_check_and_write(tmp_path):
    U = _thin_lex(L, 48)
    path = str(tmp_path / "cfg.oqcd")
    blob = bytearray(_openqcd_bytes(L, U))
    blob[24 + 8 * 18 * 8 * 7 + 6] ^= 0x08                                          # damage one link: the plaquette no longer matches
    open(path, "wb").write(bytes(blob))
    with pytest.raises(binding.HisqError) as e:
        binding.cfg_read(path, "openqcd")
    assert e.value.code == binding.HISQ_EIO
    open(path, "wb").write(_openqcd_bytes(L, U)[:-64])
    with pytest.raises(binding.HisqError):
        binding.cfg_read(path, "openqcd")
    out = str(tmp_path / "out.oqcd")
    binding.cfg_write(out, "openqcd", torch.from_numpy(_canonical(L, U)), L, real_bytes=8)
    mine, theirs = open(out, "rb").read(), _openqcd_bytes(L, U)
    assert mine[:16] == theirs[:16] and mine[24:] == theirs[24:]                    # sizes and every link, bit for bit
    assert abs(struct.unpack("<d", mine[16:24])[0] - struct.unpack("<d", theirs[16:24])[0]) < 1e-12
    with pytest.raises(binding.HisqError):
        binding.cfg_write(out, "openqcd", torch.from_numpy(_canonical(L, U)), L, real_bytes=4)
