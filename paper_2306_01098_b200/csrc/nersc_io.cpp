// nersc_io.cpp -- host-side reader / writer of gauge configurations in the NERSC archive format (
// PAPER.md:540 lists "ILDG, MILC, NERSC, openQCD" among the formats the paper's code reads).  Plain C++ on host memory:
// the caller copies the result to the device and hands it to hisq_smear.  No CUDA in this file.
//
// The format (public, text header + raw binary): a header of `KEY = VALUE` lines between BEGIN_HEADER and END_HEADER with
//   DATATYPE = 4D_SU3_GAUGE_3x3 (all three rows stored) | 4D_SU3_GAUGE (rows 0, 1; row 2 = conj(row0 x row1))
//   DIMENSION_1..4 = Lx, Ly, Lz, Lt        FLOATING_POINT = IEEE64BIG | IEEE32BIG | IEEE64LITTLE | IEEE32LITTLE
//   CHECKSUM = hex: sum modulo 2^32 of all 32-bit words of the data (in the file's declared byte order)
//   LINK_TRACE = mean of Re tr U / 3       PLAQUETTE = mean of Re tr U_plaq / 3 (verified when the header gives a non-zero value)
// followed by the links, site by site with x fastest (the lexicographic order of PAPER.md:433), and for each site
// mu = 0..3, each matrix row-major (re, im).  The result goes to the CANONICAL layout of include/hisq.h (Eq. (5):
// slot mu*V + eo(x)) as complex double.
#include "../../include/hisq.h"

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

double hisq_host_plaquette(const int* L, const double* links);   // cfg_io.cpp

namespace {

struct Header {
    int L[4] = { 0, 0, 0, 0 };
    bool rows3 = true, f64 = true, big = true;
    uint32_t checksum = 0;
    double link_trace = 0.0, plaquette = 0.0;
    bool have_checksum = false, have_type = false, have_fp = false, have_link_trace = false, have_plaquette = false;
    long data_offset = 0;
};

std::string trim(const std::string& s)
{
    size_t a = s.find_first_not_of(" \t\r\n"), b = s.find_last_not_of(" \t\r\n");
    return a == std::string::npos ? std::string() : s.substr(a, b - a + 1);
}

// 0 ok, HISQ_EIO unreadable, HISQ_EINVAL malformed
int read_header(FILE* f, Header& h)
{
    char line[1024];
    if (!fgets(line, sizeof line, f) || trim(line) != "BEGIN_HEADER") return HISQ_EINVAL;
    bool ended = false;
    while (fgets(line, sizeof line, f)) {
        const std::string s = trim(line);
        if (s == "END_HEADER") { ended = true; break; }
        const size_t eq = s.find('=');
        if (eq == std::string::npos) continue;
        const std::string key = trim(s.substr(0, eq)), val = trim(s.substr(eq + 1));
        if (key == "DATATYPE") {
            if (val == "4D_SU3_GAUGE_3x3") h.rows3 = true;
            else if (val == "4D_SU3_GAUGE") h.rows3 = false;
            else return HISQ_EINVAL;
            h.have_type = true;
        } else if (key.rfind("DIMENSION_", 0) == 0 && key.size() == 11 && key[10] >= '1' && key[10] <= '4') {
            h.L[key[10] - '1'] = atoi(val.c_str());
        } else if (key == "CHECKSUM") {
            h.checksum = (uint32_t)strtoul(val.c_str(), nullptr, 16);
            h.have_checksum = true;
        } else if (key == "LINK_TRACE") { h.link_trace = atof(val.c_str()); h.have_link_trace = true; }
        else if (key == "PLAQUETTE") { h.plaquette = atof(val.c_str()); h.have_plaquette = true; }
        else if (key.rfind("BOUNDARY_", 0) == 0) {
            if (val != "PERIODIC") return HISQ_EINVAL;   // the library's gauge field is periodic
        }
        else if (key == "FLOATING_POINT") {
            if (val == "IEEE64BIG") { h.f64 = true; h.big = true; }
            else if (val == "IEEE32BIG" || val == "IEEE32") { h.f64 = false; h.big = true; }
            else if (val == "IEEE64LITTLE") { h.f64 = true; h.big = false; }
            else if (val == "IEEE32LITTLE") { h.f64 = false; h.big = false; }
            else return HISQ_EINVAL;
            h.have_fp = true;
        }
    }
    if (!ended || !h.have_type || !h.have_fp) return HISQ_EINVAL;
    for (int d = 0; d < 4; ++d)
        if (h.L[d] < 1 || h.L[d] > 4096) return HISQ_EINVAL;
    h.data_offset = ftell(f);
    return HISQ_OK;
}

inline uint32_t load32(const unsigned char* p, bool big)
{
    return big ? ((uint32_t)p[0] << 24) | ((uint32_t)p[1] << 16) | ((uint32_t)p[2] << 8) | (uint32_t)p[3]
               : ((uint32_t)p[3] << 24) | ((uint32_t)p[2] << 16) | ((uint32_t)p[1] << 8) | (uint32_t)p[0];
}
inline void store32(unsigned char* p, uint32_t v)   // big-endian
{
    p[0] = (unsigned char)(v >> 24); p[1] = (unsigned char)(v >> 16); p[2] = (unsigned char)(v >> 8); p[3] = (unsigned char)v;
}

inline size_t canonical_slot(const int* L, size_t lex, int mu)
{
    const size_t V = (size_t)L[0] * L[1] * L[2] * L[3];
    const int x = (int)(lex % L[0]), y = (int)((lex / L[0]) % L[1]), z = (int)((lex / ((size_t)L[0] * L[1])) % L[2]),
              t = (int)(lex / ((size_t)L[0] * L[1] * L[2]));
    return (size_t)mu * V + lex / 2 + (size_t)((x + y + z + t) & 1) * (V / 2);
}

}  // namespace

extern "C" int hisq_nersc_info(const char* path, int* L, int* rows, int* real_bytes, double* link_trace, double* plaquette)
{
    if (!path) return HISQ_EINVAL;
    FILE* f = fopen(path, "rb");
    if (!f) return HISQ_EIO;
    Header h;
    const int rc = read_header(f, h);
    fclose(f);
    if (rc) return rc;
    if (L) for (int d = 0; d < 4; ++d) L[d] = h.L[d];
    if (rows) *rows = h.rows3 ? 3 : 2;
    if (real_bytes) *real_bytes = h.f64 ? 8 : 4;
    if (link_trace) *link_trace = h.link_trace;
    if (plaquette) *plaquette = h.plaquette;
    return HISQ_OK;
}

extern "C" int hisq_nersc_read(const char* path, void* links_host, size_t bytes)
{
    if (!path || !links_host) return HISQ_EINVAL;
    FILE* f = fopen(path, "rb");
    if (!f) return HISQ_EIO;
    Header h;
    int rc = read_header(f, h);
    if (rc) { fclose(f); return rc; }
    for (int d = 0; d < 4; ++d)
        if (h.L[d] < 4 || (h.L[d] & 1)) { fclose(f); return HISQ_EINVAL; }   // the library's lattices: even extents >= 4
    const size_t V = (size_t)h.L[0] * h.L[1] * h.L[2] * h.L[3];
    if (bytes < V * 4 * 18 * sizeof(double)) { fclose(f); return HISQ_EINVAL; }
    const int nreal = h.rows3 ? 18 : 12, w = h.f64 ? 8 : 4;
    const size_t site_bytes = (size_t)4 * nreal * w;
    std::vector<unsigned char> buf(site_bytes);
    double* out = (double*)links_host;
    uint32_t sum = 0;
    double trace = 0.0;
    for (size_t lex = 0; lex < V; ++lex) {
        if (fread(buf.data(), 1, site_bytes, f) != site_bytes) { fclose(f); return HISQ_EIO; }
        for (size_t i = 0; i < site_bytes; i += 4) sum += load32(&buf[i], h.big);
        for (int mu = 0; mu < 4; ++mu) {
            double m[18];
            const unsigned char* p = &buf[(size_t)mu * nreal * w];
            for (int e = 0; e < nreal; ++e) {
                if (h.f64) {
                    const uint32_t a = load32(p + 8 * e, h.big), b = load32(p + 8 * e + 4, h.big);
                    const uint64_t u = h.big ? ((uint64_t)a << 32) | b : ((uint64_t)b << 32) | a;
                    memcpy(&m[e], &u, 8);
                } else {
                    const uint32_t a = load32(p + 4 * e, h.big);
                    float v;
                    memcpy(&v, &a, 4);
                    m[e] = v;
                }
            }
            if (!h.rows3) {   // row 2 = conj(row 0 x row 1)
                for (int a = 0; a < 3; ++a) {
                    const int b = (a + 1) % 3, c = (a + 2) % 3;
                    const double re = (m[2 * b] * m[6 + 2 * c] - m[2 * b + 1] * m[6 + 2 * c + 1]) - (m[2 * c] * m[6 + 2 * b] - m[2 * c + 1] * m[6 + 2 * b + 1]);
                    const double im = (m[2 * b] * m[6 + 2 * c + 1] + m[2 * b + 1] * m[6 + 2 * c]) - (m[2 * c] * m[6 + 2 * b + 1] + m[2 * c + 1] * m[6 + 2 * b]);
                    m[12 + 2 * a] = re;
                    m[12 + 2 * a + 1] = -im;
                }
            }
            trace += m[0] + m[8] + m[16];
            memcpy(out + canonical_slot(h.L, lex, mu) * 18, m, sizeof m);
        }
    }
    fclose(f);
    if (!h.have_checksum) return HISQ_EINVAL;               // a file without its checksum cannot be trusted
    if (sum != h.checksum) return HISQ_EIO;
    const double lt = trace / (3.0 * 4.0 * (double)V);
    if (h.have_link_trace && std::fabs(lt - h.link_trace) > 1e-5 * (1.0 + std::fabs(h.link_trace))) return HISQ_EIO;
    // the header's plaquette (mean Re tr / 3 over the 6 planes); writers that do not know it put 0: not checked then
    if (h.have_plaquette && h.plaquette != 0.0 &&
        std::fabs(hisq_host_plaquette(h.L, out) / 3.0 - h.plaquette) > 1e-5 * (1.0 + std::fabs(h.plaquette)))
        return HISQ_EIO;
    return HISQ_OK;
}

extern "C" int hisq_nersc_write(const char* path, const void* links_host, const int* L, int rows, double plaquette)
{
    if (!path || !links_host || !L || (rows != 2 && rows != 3)) return HISQ_EINVAL;
    for (int d = 0; d < 4; ++d)
        if (L[d] < 4 || (L[d] & 1)) return HISQ_EINVAL;
    const size_t V = (size_t)L[0] * L[1] * L[2] * L[3];
    const int nreal = rows == 3 ? 18 : 12;
    const double* in = (const double*)links_host;
    std::vector<unsigned char> data(V * 4 * nreal * 8);
    uint32_t sum = 0;
    double trace = 0.0;
    size_t o = 0;
    for (size_t lex = 0; lex < V; ++lex)
        for (int mu = 0; mu < 4; ++mu) {
            const double* m = in + canonical_slot(L, lex, mu) * 18;
            trace += m[0] + m[8] + m[16];
            for (int e = 0; e < nreal; ++e) {
                uint64_t u;
                memcpy(&u, &m[e], 8);
                store32(&data[o], (uint32_t)(u >> 32)); store32(&data[o + 4], (uint32_t)u);
                sum += (uint32_t)(u >> 32); sum += (uint32_t)u;
                o += 8;
            }
        }
    FILE* f = fopen(path, "wb");
    if (!f) return HISQ_EIO;
    fprintf(f, "BEGIN_HEADER\nHDR_VERSION = 1.0\nDATATYPE = %s\nSTORAGE_FORMAT = 1.0\n", rows == 3 ? "4D_SU3_GAUGE_3x3" : "4D_SU3_GAUGE");
    for (int d = 0; d < 4; ++d) fprintf(f, "DIMENSION_%d = %d\n", d + 1, L[d]);
    fprintf(f, "LINK_TRACE = %.12f\nPLAQUETTE = %.12f\n", trace / (12.0 * (double)V), plaquette);
    for (int d = 0; d < 4; ++d) fprintf(f, "BOUNDARY_%d = PERIODIC\n", d + 1);
    fprintf(f, "CHECKSUM = %x\nFLOATING_POINT = IEEE64BIG\nEND_HEADER\n", sum);
    const bool ok = fwrite(data.data(), 1, data.size(), f) == data.size();
    return (fclose(f) == 0 && ok) ? HISQ_OK : HISQ_EIO;
}
