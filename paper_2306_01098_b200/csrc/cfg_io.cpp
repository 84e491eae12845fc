// cfg_io.cpp -- host-side readers / writers of gauge configurations in the ILDG, MILC (version 5) and openQCD formats
// (the paper's code "supports the ILDG format", MILC, NERSC and openQCD).  The NERSC
// format is nersc_io.cpp.  Plain C++ on host memory, no CUDA: the caller copies the CANONICAL link array (include/hisq.h,
// Eq. (5): matrix of (x, mu) at slot mu*V + eo(x), 9 complex doubles row-major) to the device and calls hisq_smear.
//
// The formats as restated here from their public descriptions (there is no archive file in this container to check
// against: the tests write files with independent numpy writers of the same descriptions):
//
// ILDG     a LIME container: records of [144-byte header: magic 0x456789ab, version (u16), flags (u16: 0x8000 message
//          begin, 0x4000 message end), payload length (u64), type (128 chars)] + payload padded to 8 bytes, all big-endian.
//          Record "ildg-format": XML with <precision>32|64</precision>, <lx> <ly> <lz> <lt>.  Record "ildg-binary-data":
//          sites with x fastest, then y, z, t; per site mu = x, y, z, t; per link 9 complex row-major, IEEE big-endian.
//          Record "scidac-checksum" (optional): XML <suma>, <sumb> (hex): with c_s = CRC-32 of the bytes of site s,
//          suma = XOR_s rotl(c_s, s mod 29), sumb = XOR_s rotl(c_s, s mod 31); verified when present.
// MILC v5  header: i32 magic 20103 (its byte order tells the file's), i32 dims[4], char time_stamp[64], i32 order (0 =
//          natural site order; anything else is refused), u32 sum29, u32 sum31; then sites with x fastest, per site
//          mu = x, y, z, t, per link 9 complex row-major of IEEE float32.  With w_k the k-th 32-bit word of the data,
//          sum29 = XOR_k rotl(w_k, k mod 29), sum31 = XOR_k rotl(w_k, k mod 31).
// openQCD  little-endian: i32 N0 (time), N1, N2, N3 (space), f64 average plaquette (3 for unit links), then for every ODD
//          point, ordered with x0 slowest and x3 fastest, the 8 links U(x,+0), U(x,-0), U(x,+1), ..., U(x,-3) where
//          U(x,-mu) is the link from x - mu to x, each 9 complex doubles row-major.  Directions 1, 2, 3 are our x, y, z and
//          0 is our t.  The plaquette is the format's only integrity check: recomputed here and compared.
#include "../../include/hisq.h"

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

namespace {

struct File {
    FILE* f;
    explicit File(const char* path, const char* mode) : f(fopen(path, mode)) {}
    ~File() { if (f) fclose(f); }
};

bool extents_ok(const int* L)
{
    for (int d = 0; d < 4; ++d)
        if (L[d] < 4 || (L[d] & 1) || L[d] > 4096) return false;   // the library's lattices: even extents >= 4
    return true;
}

inline size_t volume(const int* L) { return (size_t)L[0] * L[1] * L[2] * L[3]; }

inline size_t lex_of(const int* L, const int* c) { return c[0] + (size_t)L[0] * (c[1] + (size_t)L[1] * (c[2] + (size_t)L[2] * c[3])); }

inline size_t canonical_slot(const int* L, size_t lex, int mu)
{
    const size_t V = volume(L);
    const int x = (int)(lex % L[0]), y = (int)((lex / L[0]) % L[1]), z = (int)((lex / ((size_t)L[0] * L[1])) % L[2]),
              t = (int)(lex / ((size_t)L[0] * L[1] * L[2]));
    return (size_t)mu * V + lex / 2 + (size_t)((x + y + z + t) & 1) * (V / 2);
}

inline uint32_t bswap32(uint32_t v) { return (v >> 24) | ((v >> 8) & 0xff00u) | ((v << 8) & 0xff0000u) | (v << 24); }
inline uint64_t bswap64(uint64_t v) { return ((uint64_t)bswap32((uint32_t)v) << 32) | bswap32((uint32_t)(v >> 32)); }
inline bool host_is_little() { const uint16_t one = 1; return *(const unsigned char*)&one == 1; }
inline uint32_t rotl(uint32_t v, unsigned r) { return r ? (v << r) | (v >> (32 - r)) : v; }

// IEEE value of `w` bytes at p in the given byte order -> double
inline double load_real(const unsigned char* p, int w, bool big)
{
    if (w == 8) {
        uint64_t u;
        memcpy(&u, p, 8);
        if (big == host_is_little()) u = bswap64(u);
        double d;
        memcpy(&d, &u, 8);
        return d;
    }
    uint32_t u;
    memcpy(&u, p, 4);
    if (big == host_is_little()) u = bswap32(u);
    float v;
    memcpy(&v, &u, 4);
    return v;
}
inline void store_real(unsigned char* p, double d, int w, bool big)
{
    if (w == 8) {
        uint64_t u;
        memcpy(&u, &d, 8);
        if (big == host_is_little()) u = bswap64(u);
        memcpy(p, &u, 8);
    } else {
        const float v = (float)d;
        uint32_t u;
        memcpy(&u, &v, 4);
        if (big == host_is_little()) u = bswap32(u);
        memcpy(p, &u, 4);
    }
}

// CRC-32 (reflected polynomial 0xEDB88320, initial value and final XOR 0xFFFFFFFF), bit by bit table built on first use
uint32_t crc32(const unsigned char* p, size_t n)
{
    static uint32_t table[256];
    static bool have = false;
    if (!have) {
        for (uint32_t i = 0; i < 256; ++i) {
            uint32_t c = i;
            for (int k = 0; k < 8; ++k) c = (c & 1) ? 0xEDB88320u ^ (c >> 1) : c >> 1;
            table[i] = c;
        }
        have = true;
    }
    uint32_t c = 0xFFFFFFFFu;
    for (size_t i = 0; i < n; ++i) c = table[(c ^ p[i]) & 0xff] ^ (c >> 8);
    return c ^ 0xFFFFFFFFu;
}

// 3x3 complex helpers on 18 doubles, row-major
inline void mat_mul(const double* a, const double* b, double* c, bool dag_b)
{
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double re = 0.0, im = 0.0;
            for (int k = 0; k < 3; ++k) {
                const double ar = a[2 * (3 * i + k)], ai = a[2 * (3 * i + k) + 1];
                const double br = dag_b ? b[2 * (3 * j + k)] : b[2 * (3 * k + j)];
                const double bi = dag_b ? -b[2 * (3 * j + k) + 1] : b[2 * (3 * k + j) + 1];
                re += ar * br - ai * bi;
                im += ar * bi + ai * br;
            }
            c[2 * (3 * i + j)] = re;
            c[2 * (3 * i + j) + 1] = im;
        }
}

}  // namespace

// mean over sites and the 6 planes of Re tr [U_mu(x) U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+] (3 for unit links), periodic;
// links: CANONICAL array.  Also used by nersc_io.cpp (the header's PLAQUETTE is this / 3).
double hisq_host_plaquette(const int* L, const double* links)
{
    const size_t V = volume(L);
    double tot = 0.0;
    int c[4];
    for (c[3] = 0; c[3] < L[3]; ++c[3])
        for (c[2] = 0; c[2] < L[2]; ++c[2])
            for (c[1] = 0; c[1] < L[1]; ++c[1])
                for (c[0] = 0; c[0] < L[0]; ++c[0]) {
                    const size_t x = lex_of(L, c);
                    for (int mu = 0; mu < 4; ++mu)
                        for (int nu = mu + 1; nu < 4; ++nu) {
                            int cm[4] = { c[0], c[1], c[2], c[3] }, cn[4] = { c[0], c[1], c[2], c[3] };
                            cm[mu] = (cm[mu] + 1) % L[mu];
                            cn[nu] = (cn[nu] + 1) % L[nu];
                            const double* a = links + canonical_slot(L, x, mu) * 18;
                            const double* b = links + canonical_slot(L, lex_of(L, cm), nu) * 18;
                            const double* d = links + canonical_slot(L, lex_of(L, cn), mu) * 18;
                            const double* e = links + canonical_slot(L, x, nu) * 18;
                            double ab[18], abd[18], p[18];
                            mat_mul(a, b, ab, false);
                            mat_mul(ab, d, abd, true);
                            mat_mul(abd, e, p, true);
                            tot += p[0] + p[8] + p[16];
                        }
                }
    return tot / (6.0 * (double)V);
}

// ---- sites in lexicographic order, mu = 0..3 per site, 9 complex row-major: the body shared by ILDG and MILC ----------
namespace {

// reads V sites of 72 reals of width w from f into the canonical array; per-site callback sees the raw bytes
template <typename PerSite>
int read_lex_body(FILE* f, const int* L, int w, bool big, double* out, PerSite per_site)
{
    const size_t V = volume(L), site_bytes = (size_t)72 * w;
    std::vector<unsigned char> buf(site_bytes);
    for (size_t lex = 0; lex < V; ++lex) {
        if (fread(buf.data(), 1, site_bytes, f) != site_bytes) return HISQ_EIO;
        per_site(lex, buf.data(), site_bytes);
        for (int mu = 0; mu < 4; ++mu) {
            double* m = out + canonical_slot(L, lex, mu) * 18;
            for (int e = 0; e < 18; ++e) m[e] = load_real(&buf[(size_t)(mu * 18 + e) * w], w, big);
        }
    }
    return HISQ_OK;
}

template <typename PerSite>
bool write_lex_body(FILE* f, const int* L, int w, bool big, const double* in, PerSite per_site)
{
    const size_t V = volume(L), site_bytes = (size_t)72 * w;
    std::vector<unsigned char> buf(site_bytes);
    for (size_t lex = 0; lex < V; ++lex) {
        for (int mu = 0; mu < 4; ++mu) {
            const double* m = in + canonical_slot(L, lex, mu) * 18;
            for (int e = 0; e < 18; ++e) store_real(&buf[(size_t)(mu * 18 + e) * w], m[e], w, big);
        }
        per_site(lex, buf.data(), site_bytes);
        if (fwrite(buf.data(), 1, site_bytes, f) != site_bytes) return false;
    }
    return true;
}

// ---- ILDG (LIME) ---------------------------------------------------------------------------------------------------------
const uint32_t kLimeMagic = 0x456789abu;
struct LimeRecord { std::string type; uint64_t length; long offset; };

// next record header at the current position; 1 = end of file, 0 = ok, < 0 = error
int lime_next(FILE* f, LimeRecord& r)
{
    unsigned char h[144];
    const size_t got = fread(h, 1, 144, f);
    if (got == 0) return 1;
    if (got != 144) return HISQ_EIO;
    const uint32_t magic = ((uint32_t)h[0] << 24) | ((uint32_t)h[1] << 16) | ((uint32_t)h[2] << 8) | h[3];
    if (magic != kLimeMagic) return HISQ_EINVAL;
    r.length = 0;
    for (int i = 0; i < 8; ++i) r.length = (r.length << 8) | h[8 + i];
    h[143] = 0;
    r.type = std::string((const char*)h + 16);
    r.offset = ftell(f);
    return 0;
}
int lime_skip(FILE* f, const LimeRecord& r)
{
    const uint64_t padded = (r.length + 7) / 8 * 8;
    return fseek(f, r.offset + (long)padded, SEEK_SET) == 0 ? 0 : HISQ_EIO;
}
bool lime_write_header(FILE* f, const char* type, uint64_t length, bool begin, bool end)
{
    unsigned char h[144];
    memset(h, 0, sizeof h);
    h[0] = 0x45; h[1] = 0x67; h[2] = 0x89; h[3] = 0xab;
    h[4] = 0; h[5] = 1;                                              // version 1
    h[6] = (unsigned char)((begin ? 0x80 : 0) | (end ? 0x40 : 0));   // flags, high byte
    for (int i = 0; i < 8; ++i) h[8 + i] = (unsigned char)(length >> (56 - 8 * i));
    strncpy((char*)h + 16, type, 127);
    return fwrite(h, 1, 144, f) == 144;
}
bool lime_pad(FILE* f, uint64_t length)
{
    const unsigned char z[8] = { 0 };
    const size_t pad = (size_t)((8 - length % 8) % 8);
    return pad == 0 || fwrite(z, 1, pad, f) == pad;
}
// text between <tag> and </tag>, "" if absent
std::string xml_field(const std::string& xml, const char* tag)
{
    const std::string open = std::string("<") + tag + ">", close = std::string("</") + tag + ">";
    const size_t a = xml.find(open);
    if (a == std::string::npos) return std::string();
    const size_t b = xml.find(close, a);
    if (b == std::string::npos) return std::string();
    return xml.substr(a + open.size(), b - a - open.size());
}

struct IldgInfo { int L[4] = { 0, 0, 0, 0 }; int w = 0; long data_offset = -1; uint64_t data_len = 0; bool have_sum = false; uint32_t suma = 0, sumb = 0; };

int ildg_scan(FILE* f, IldgInfo& info)
{
    LimeRecord r;
    int rc;
    while ((rc = lime_next(f, r)) == 0) {
        if (r.type == "ildg-format" || r.type == "scidac-checksum") {
            if (r.length > (1u << 20)) return HISQ_EINVAL;
            std::string xml((size_t)r.length, '\0');
            if (fread(&xml[0], 1, (size_t)r.length, f) != r.length) return HISQ_EIO;
            if (r.type == "ildg-format") {
                if (xml_field(xml, "field").find("su3gauge") == std::string::npos) return HISQ_EINVAL;
                const int prec = atoi(xml_field(xml, "precision").c_str());
                if (prec != 32 && prec != 64) return HISQ_EINVAL;
                info.w = prec / 8;
                const char* tags[4] = { "lx", "ly", "lz", "lt" };
                for (int d = 0; d < 4; ++d) info.L[d] = atoi(xml_field(xml, tags[d]).c_str());
            } else {
                const std::string a = xml_field(xml, "suma"), b = xml_field(xml, "sumb");
                if (!a.empty() && !b.empty()) {
                    info.suma = (uint32_t)strtoul(a.c_str(), nullptr, 16);
                    info.sumb = (uint32_t)strtoul(b.c_str(), nullptr, 16);
                    info.have_sum = true;
                }
            }
        } else if (r.type == "ildg-binary-data") {
            info.data_offset = r.offset;
            info.data_len = r.length;
        }
        if ((rc = lime_skip(f, r)) != 0) return rc;
    }
    if (rc < 0) return rc;
    if (info.w == 0 || info.data_offset < 0) return HISQ_EINVAL;
    for (int d = 0; d < 4; ++d)
        if (info.L[d] < 1 || info.L[d] > 4096) return HISQ_EINVAL;
    if (info.data_len != (uint64_t)volume(info.L) * 72 * info.w) return HISQ_EINVAL;
    return HISQ_OK;
}

int ildg_read(const char* path, double* out, size_t bytes)
{
    File fl(path, "rb");
    if (!fl.f) return HISQ_EIO;
    IldgInfo info;
    int rc = ildg_scan(fl.f, info);
    if (rc) return rc;
    if (!extents_ok(info.L)) return HISQ_EINVAL;
    if (bytes < volume(info.L) * 72 * sizeof(double)) return HISQ_EINVAL;
    if (fseek(fl.f, info.data_offset, SEEK_SET) != 0) return HISQ_EIO;
    uint32_t suma = 0, sumb = 0;
    rc = read_lex_body(fl.f, info.L, info.w, true, out, [&](size_t lex, const unsigned char* p, size_t n) {
        const uint32_t c = crc32(p, n);
        suma ^= rotl(c, (unsigned)(lex % 29));
        sumb ^= rotl(c, (unsigned)(lex % 31));
    });
    if (rc) return rc;
    if (info.have_sum && (suma != info.suma || sumb != info.sumb)) return HISQ_EIO;
    return HISQ_OK;
}

int ildg_write(const char* path, const double* in, const int* L, int w)
{
    File fl(path, "wb");
    if (!fl.f) return HISQ_EIO;
    char xml[512];
    const int n = snprintf(xml, sizeof xml,
                           "<?xml version=\"1.0\" encoding=\"UTF-8\"?><ildgFormat xmlns=\"http://www.lqcd.org/ildg\"><version>1.0</version>"
                           "<field>su3gauge</field><precision>%d</precision><lx>%d</lx><ly>%d</ly><lz>%d</lz><lt>%d</lt></ildgFormat>",
                           8 * w, L[0], L[1], L[2], L[3]);
    bool ok = lime_write_header(fl.f, "ildg-format", (uint64_t)n, true, false) && fwrite(xml, 1, (size_t)n, fl.f) == (size_t)n &&
              lime_pad(fl.f, (uint64_t)n);
    const uint64_t len = (uint64_t)volume(L) * 72 * w;
    ok = ok && lime_write_header(fl.f, "ildg-binary-data", len, false, false);
    uint32_t suma = 0, sumb = 0;
    ok = ok && write_lex_body(fl.f, L, w, true, in, [&](size_t lex, const unsigned char* p, size_t nb) {
             const uint32_t c = crc32(p, nb);
             suma ^= rotl(c, (unsigned)(lex % 29));
             sumb ^= rotl(c, (unsigned)(lex % 31));
         });
    ok = ok && lime_pad(fl.f, len);
    char cs[256];
    const int m = snprintf(cs, sizeof cs, "<?xml version=\"1.0\" encoding=\"UTF-8\"?><scidacChecksum><version>1.0</version><suma>%08x</suma><sumb>%08x</sumb></scidacChecksum>",
                           suma, sumb);
    ok = ok && lime_write_header(fl.f, "scidac-checksum", (uint64_t)m, false, true) && fwrite(cs, 1, (size_t)m, fl.f) == (size_t)m &&
         lime_pad(fl.f, (uint64_t)m);
    return ok ? HISQ_OK : HISQ_EIO;
}

// ---- MILC version 5 -----------------------------------------------------------------------------------------------------
const int32_t kMilcMagic = 20103;
struct MilcInfo { int L[4]; bool swap; uint32_t sum29, sum31; };

int milc_header(FILE* f, MilcInfo& h)
{
    unsigned char b[96];
    if (fread(b, 1, 96, f) != 96) return HISQ_EIO;
    uint32_t w[24];
    memcpy(w, b, 96);
    h.swap = false;
    if ((int32_t)w[0] != kMilcMagic) {
        if ((int32_t)bswap32(w[0]) != kMilcMagic) return HISQ_EINVAL;
        h.swap = true;
    }
    auto word = [&](int i) { return h.swap ? bswap32(w[i]) : w[i]; };
    for (int d = 0; d < 4; ++d) {
        h.L[d] = (int32_t)word(1 + d);
        if (h.L[d] < 1 || h.L[d] > 4096) return HISQ_EINVAL;
    }
    if ((int32_t)word(21) != 0) return HISQ_EINVAL;   // order: only the natural site order (no site list) is read
    h.sum29 = word(22);
    h.sum31 = word(23);
    return HISQ_OK;
}

int milc_read(const char* path, double* out, size_t bytes)
{
    File fl(path, "rb");
    if (!fl.f) return HISQ_EIO;
    MilcInfo h;
    int rc = milc_header(fl.f, h);
    if (rc) return rc;
    if (!extents_ok(h.L)) return HISQ_EINVAL;
    if (bytes < volume(h.L) * 72 * sizeof(double)) return HISQ_EINVAL;
    const bool big = h.swap ? host_is_little() : !host_is_little();   // the file's byte order
    uint32_t s29 = 0, s31 = 0;
    rc = read_lex_body(fl.f, h.L, 4, big, out, [&](size_t lex, const unsigned char* p, size_t n) {
        uint64_t k = (uint64_t)lex * 72;
        for (size_t i = 0; i < n; i += 4, ++k) {
            uint32_t v;
            memcpy(&v, p + i, 4);
            if (h.swap) v = bswap32(v);
            s29 ^= rotl(v, (unsigned)(k % 29));
            s31 ^= rotl(v, (unsigned)(k % 31));
        }
    });
    if (rc) return rc;
    return (s29 == h.sum29 && s31 == h.sum31) ? HISQ_OK : HISQ_EIO;
}

int milc_write(const char* path, const double* in, const int* L)
{
    File fl(path, "wb");
    if (!fl.f) return HISQ_EIO;
    unsigned char hdr[96];
    memset(hdr, 0, sizeof hdr);
    int32_t w[5] = { kMilcMagic, L[0], L[1], L[2], L[3] };
    memcpy(hdr, w, 20);
    strncpy((char*)hdr + 20, "written by libhisq (synthetic)", 63);
    if (fwrite(hdr, 1, 96, fl.f) != 96) return HISQ_EIO;          // order = 0; the checksums are patched in below
    uint32_t s29 = 0, s31 = 0;
    const bool ok = write_lex_body(fl.f, L, 4, !host_is_little(), in, [&](size_t lex, const unsigned char* p, size_t n) {
        uint64_t k = (uint64_t)lex * 72;
        for (size_t i = 0; i < n; i += 4, ++k) {
            uint32_t v;
            memcpy(&v, p + i, 4);
            s29 ^= rotl(v, (unsigned)(k % 29));
            s31 ^= rotl(v, (unsigned)(k % 31));
        }
    });
    if (!ok || fseek(fl.f, 88, SEEK_SET) != 0) return HISQ_EIO;
    const uint32_t sums[2] = { s29, s31 };
    return fwrite(sums, 4, 2, fl.f) == 2 ? HISQ_OK : HISQ_EIO;
}

}  // namespace

// ---- openQCD ---------------------------------------------------------------------------------------------------------------
namespace {

struct OqInfo { int L[4]; double plaq; };   // L in OUR order (x, y, z, t)

int oq_header(FILE* f, OqInfo& h)
{
    unsigned char b[24];
    if (fread(b, 1, 24, f) != 24) return HISQ_EIO;
    int32_t n[4];
    for (int i = 0; i < 4; ++i) {
        uint32_t u;
        memcpy(&u, b + 4 * i, 4);
        if (!host_is_little()) u = bswap32(u);
        n[i] = (int32_t)u;
        if (n[i] < 1 || n[i] > 4096) return HISQ_EINVAL;
    }
    h.L[0] = n[1]; h.L[1] = n[2]; h.L[2] = n[3]; h.L[3] = n[0];
    h.plaq = load_real(b + 16, 8, false);
    return HISQ_OK;
}

// visits the odd points in file order; fn(our coordinates c[4]) handles the 8 matrices of one point
template <typename Fn> int oq_for_odd_points(const int* L, Fn fn)
{
    int c[4];
    for (c[3] = 0; c[3] < L[3]; ++c[3])            // x0 = t, slowest
        for (c[0] = 0; c[0] < L[0]; ++c[0])        // x1 = x
            for (c[1] = 0; c[1] < L[1]; ++c[1])    // x2 = y
                for (c[2] = 0; c[2] < L[2]; ++c[2]) {   // x3 = z, fastest
                    if (((c[0] + c[1] + c[2] + c[3]) & 1) == 0) continue;
                    const int rc = fn(c);
                    if (rc) return rc;
                }
    return HISQ_OK;
}

int oq_read(const char* path, double* out, size_t bytes)
{
    File fl(path, "rb");
    if (!fl.f) return HISQ_EIO;
    OqInfo h;
    int rc = oq_header(fl.f, h);
    if (rc) return rc;
    if (!extents_ok(h.L)) return HISQ_EINVAL;
    if (bytes < volume(h.L) * 72 * sizeof(double)) return HISQ_EINVAL;
    unsigned char buf[8 * 18 * 8];
    rc = oq_for_odd_points(h.L, [&](const int* c) {
        if (fread(buf, 1, sizeof buf, fl.f) != sizeof buf) return (int)HISQ_EIO;
        for (int mo = 0; mo < 4; ++mo) {
            const int mu = (mo + 3) % 4;               // openQCD direction 0 is time
            int cb[4] = { c[0], c[1], c[2], c[3] };
            cb[mu] = (cb[mu] - 1 + h.L[mu]) % h.L[mu];
            double* fw = out + canonical_slot(h.L, lex_of(h.L, c), mu) * 18;    // U(x, +mu): the link leaving the odd point
            double* bw = out + canonical_slot(h.L, lex_of(h.L, cb), mu) * 18;   // U(x, -mu): the link from x - mu to x
            for (int e = 0; e < 18; ++e) {
                fw[e] = load_real(buf + (size_t)((2 * mo) * 18 + e) * 8, 8, false);
                bw[e] = load_real(buf + (size_t)((2 * mo + 1) * 18 + e) * 8, 8, false);
            }
        }
        return (int)HISQ_OK;
    });
    if (rc) return rc;
    const double p = hisq_host_plaquette(h.L, out);
    return std::fabs(p - h.plaq) <= 1e-9 * (1.0 + std::fabs(h.plaq)) ? HISQ_OK : HISQ_EIO;
}

int oq_write(const char* path, const double* in, const int* L)
{
    File fl(path, "wb");
    if (!fl.f) return HISQ_EIO;
    unsigned char hdr[24];
    const int32_t n[4] = { L[3], L[0], L[1], L[2] };
    for (int i = 0; i < 4; ++i) {
        uint32_t u = (uint32_t)n[i];
        if (!host_is_little()) u = bswap32(u);
        memcpy(hdr + 4 * i, &u, 4);
    }
    store_real(hdr + 16, hisq_host_plaquette(L, in), 8, false);
    if (fwrite(hdr, 1, 24, fl.f) != 24) return HISQ_EIO;
    unsigned char buf[8 * 18 * 8];
    return oq_for_odd_points(L, [&](const int* c) {
        for (int mo = 0; mo < 4; ++mo) {
            const int mu = (mo + 3) % 4;
            int cb[4] = { c[0], c[1], c[2], c[3] };
            cb[mu] = (cb[mu] - 1 + L[mu]) % L[mu];
            const double* fw = in + canonical_slot(L, lex_of(L, c), mu) * 18;
            const double* bw = in + canonical_slot(L, lex_of(L, cb), mu) * 18;
            for (int e = 0; e < 18; ++e) {
                store_real(buf + (size_t)((2 * mo) * 18 + e) * 8, fw[e], 8, false);
                store_real(buf + (size_t)((2 * mo + 1) * 18 + e) * 8, bw[e], 8, false);
            }
        }
        return fwrite(buf, 1, sizeof buf, fl.f) == sizeof buf ? (int)HISQ_OK : (int)HISQ_EIO;
    });
}

}  // namespace

// ---- C ABI (include/hisq.h) ----------------------------------------------------------------------------------------------
extern "C" int hisq_cfg_info(const char* path, int format, int* L, int* real_bytes)
{
    if (!path) return HISQ_EINVAL;
    File fl(path, "rb");
    if (!fl.f) return HISQ_EIO;
    int dims[4] = { 0, 0, 0, 0 }, w = 0, rc;
    if (format == HISQ_FMT_ILDG) {
        IldgInfo i;
        if ((rc = ildg_scan(fl.f, i)) != 0) return rc;
        memcpy(dims, i.L, sizeof dims); w = i.w;
    } else if (format == HISQ_FMT_MILC) {
        MilcInfo m;
        if ((rc = milc_header(fl.f, m)) != 0) return rc;
        memcpy(dims, m.L, sizeof dims); w = 4;
    } else if (format == HISQ_FMT_OPENQCD) {
        OqInfo o;
        if ((rc = oq_header(fl.f, o)) != 0) return rc;
        memcpy(dims, o.L, sizeof dims); w = 8;
    } else return HISQ_EINVAL;
    if (L) memcpy(L, dims, sizeof dims);
    if (real_bytes) *real_bytes = w;
    return HISQ_OK;
}

extern "C" int hisq_cfg_read(const char* path, int format, void* links_host, size_t bytes)
{
    if (!path || !links_host) return HISQ_EINVAL;
    switch (format) {
    case HISQ_FMT_ILDG: return ildg_read(path, (double*)links_host, bytes);
    case HISQ_FMT_MILC: return milc_read(path, (double*)links_host, bytes);
    case HISQ_FMT_OPENQCD: return oq_read(path, (double*)links_host, bytes);
    default: return HISQ_EINVAL;
    }
}

extern "C" int hisq_cfg_write(const char* path, int format, const void* links_host, const int* L, int real_bytes)
{
    if (!path || !links_host || !L || !extents_ok(L)) return HISQ_EINVAL;
    switch (format) {
    case HISQ_FMT_ILDG: return (real_bytes == 4 || real_bytes == 8) ? ildg_write(path, (const double*)links_host, L, real_bytes) : HISQ_EINVAL;
    case HISQ_FMT_MILC: return real_bytes == 4 ? milc_write(path, (const double*)links_host, L) : HISQ_EINVAL;
    case HISQ_FMT_OPENQCD: return real_bytes == 8 ? oq_write(path, (const double*)links_host, L) : HISQ_EINVAL;
    default: return HISQ_EINVAL;
    }
}
