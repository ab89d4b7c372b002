// lhapdf_io.cu -- host-only front-end for grids stored in the LHAPDF6 text layout that PDFFlow
// reads ("the PDF data is stored in ... grids", "the (alpha_s(Q), Q) nodes
// stored in the PDF metadata file").  No device code: the parsed arrays are
// handed to pdf_grid_load / pdf_set_load / alphas_grid_load by the caller.
//
// Member file ("lhagrid1"): a metadata header, then blocks separated by lines "---".  A block is
//   line 1: the x knots;  line 2: the Q knots (GeV);  line 3: the PIDs;
//   then nx*nq lines of n_pid values, x index outer, Q index inner  (= pdf_grid_load's order).
// Metadata file: "Key: value" lines; the two lists AlphaS_Qs and AlphaS_Vals may span lines.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "pdfb_internal.cuh"

struct pdfb_lhagrid {
    int n_sub = 0, nx = 0, n_pid = 0;  // nx: knots of the first block's x array
    bool shared_x = true;              // every block carries the same x-knot array
    std::vector<double> x, q, values;  // x: the blocks' x arrays, q and values: concatenated over the blocks
    std::vector<int> x_off, q_off, pids;
};

static bool read_all(const char *path, std::string &s)
{
    FILE *f = fopen(path, "rb");
    if (!f) return false;
    char buf[1 << 16];
    size_t n;
    while ((n = fread(buf, 1, sizeof buf, f)) > 0) s.append(buf, n);
    fclose(f);
    return true;
}

// numbers of one text line; false on a token that is not a number
static bool parse_doubles(const char *b, const char *e, std::vector<double> &out)
{
    out.clear();
    std::string line(b, e);
    const char *p = line.c_str();
    for (;;) {
        while (*p == ' ' || *p == '\t' || *p == '\r' || *p == ',') ++p;
        if (!*p) return true;
        char *end = nullptr;
        double v = strtod(p, &end);
        if (end == p) return false;
        out.push_back(v);
        p = end;
    }
}

extern "C" int pdfb_lhagrid_read(const char *path, pdfb_lhagrid **out)
{
    if (!out) return PDFB_EINVAL;
    *out = nullptr;
    if (!path) return PDFB_EINVAL;
    std::string s;
    if (!read_all(path, s)) return PDFB_EIO;
    // split into lines
    std::vector<std::pair<const char *, const char *>> lines;
    for (const char *p = s.data(), *e = s.data() + s.size(); p < e;) {
        const char *nl = (const char *)memchr(p, '\n', e - p);
        const char *le = nl ? nl : e;
        lines.emplace_back(p, le);
        p = nl ? nl + 1 : e;
    }
    auto is_sep = [](const std::pair<const char *, const char *> &l) {
        const char *b = l.first, *e = l.second;
        while (e > b && (e[-1] == ' ' || e[-1] == '\r' || e[-1] == '\t')) --e;
        return e - b == 3 && b[0] == '-' && b[1] == '-' && b[2] == '-';
    };
    auto is_blank = [](const std::pair<const char *, const char *> &l) {
        for (const char *p = l.first; p < l.second; ++p) if (*p != ' ' && *p != '\r' && *p != '\t') return false;
        return true;
    };
    pdfb_lhagrid *g = new (std::nothrow) pdfb_lhagrid();
    if (!g) return PDFB_EINVAL;
    size_t i = 0;
    while (i < lines.size() && !is_sep(lines[i])) ++i;  // metadata header
    if (i == lines.size()) { delete g; return PDFB_EFORMAT; }
    ++i;
    std::vector<double> row, xk, qk;
    int rc = PDFB_OK;
    bool mixed_pids = false;  // blocks with different PID lists: parsed to the end, then refused as such
    std::vector<double> x0;
    g->q_off.push_back(0);
    while (i < lines.size() && !rc) {
        while (i < lines.size() && is_blank(lines[i])) ++i;
        if (i == lines.size()) break;  // trailing separator
        if (i + 3 > lines.size()) { rc = PDFB_EFORMAT; break; }
        if (!parse_doubles(lines[i].first, lines[i].second, xk) || !parse_doubles(lines[i + 1].first, lines[i + 1].second, qk) ||
            !parse_doubles(lines[i + 2].first, lines[i + 2].second, row)) { rc = PDFB_EFORMAT; break; }
        i += 3;
        if (xk.size() < 2 || qk.size() < 2 || row.empty()) { rc = PDFB_EFORMAT; break; }
        std::vector<int> pids(row.size());
        for (size_t k = 0; k < row.size(); k++) pids[k] = (int)row[k];
        if (g->n_sub == 0) {
            x0 = xk; g->nx = (int)xk.size(); g->pids = pids; g->n_pid = (int)pids.size();
            g->x_off.push_back(0);
        } else {
            if (pids != g->pids) mixed_pids = true;  // one PID list for all sub-grids
            if (xk != x0) g->shared_x = false;       // own x knots per sub-grid: pdf_grid_load_xs
        }
        g->x.insert(g->x.end(), xk.begin(), xk.end());
        g->x_off.push_back((int)g->x.size());
        const size_t nrows = xk.size() * qk.size();
        for (size_t r = 0; r < nrows && !rc; r++, i++) {
            if (i >= lines.size() || is_sep(lines[i]) || !parse_doubles(lines[i].first, lines[i].second, row) ||
                row.size() != pids.size()) { rc = PDFB_EFORMAT; break; }
            if (!mixed_pids) g->values.insert(g->values.end(), row.begin(), row.end());
        }
        if (rc) break;
        g->q.insert(g->q.end(), qk.begin(), qk.end());
        g->q_off.push_back((int)g->q.size());
        g->n_sub++;
        while (i < lines.size() && is_blank(lines[i])) ++i;
        if (i < lines.size()) {
            if (!is_sep(lines[i])) { rc = PDFB_EFORMAT; break; }
            ++i;
        }
    }
    if (!rc && g->n_sub == 0) rc = PDFB_EFORMAT;
    if (!rc && mixed_pids) rc = PDFB_EXKNOTS;
    if (!rc && g->n_sub > PDFB_MAX_SUBGRIDS) rc = PDFB_ELIMIT;
    if (rc) { delete g; return rc; }
    *out = g;
    return PDFB_OK;
}

extern "C" int pdfb_lhagrid_dims(const pdfb_lhagrid *g, int *n_sub, int *nx, int *nq_tot, int *n_pid)
{
    if (!g || !n_sub || !nx || !nq_tot || !n_pid) return PDFB_EINVAL;
    if (!g->shared_x) return PDFB_EXKNOTS;  // own x knots per sub-grid: pdfb_lhagrid_dims_xs / _get_xs
    *n_sub = g->n_sub; *nx = g->nx; *nq_tot = (int)g->q.size(); *n_pid = g->n_pid;
    return PDFB_OK;
}

extern "C" int pdfb_lhagrid_get(const pdfb_lhagrid *g, double *x_knots, int *q_offsets, double *q_knots, int *pids,
                                double *values)
{
    if (!g || !x_knots || !q_offsets || !q_knots || !pids || !values) return PDFB_EINVAL;
    if (!g->shared_x) return PDFB_EXKNOTS;
    memcpy(x_knots, g->x.data(), sizeof(double) * g->nx);
    memcpy(q_offsets, g->q_off.data(), sizeof(int) * g->q_off.size());
    memcpy(q_knots, g->q.data(), sizeof(double) * g->q.size());
    memcpy(pids, g->pids.data(), sizeof(int) * g->pids.size());
    memcpy(values, g->values.data(), sizeof(double) * g->values.size());
    return PDFB_OK;
}

extern "C" int pdfb_lhagrid_dims_xs(const pdfb_lhagrid *g, int *n_sub, int *nx_total, int *nq_tot, int *n_pid,
                                    long long *n_values, int *shared_x)
{
    if (!g || !n_sub || !nx_total || !nq_tot || !n_pid || !n_values || !shared_x) return PDFB_EINVAL;
    *n_sub = g->n_sub; *nx_total = (int)g->x.size(); *nq_tot = (int)g->q.size(); *n_pid = g->n_pid;
    *n_values = (long long)g->values.size(); *shared_x = g->shared_x ? 1 : 0;
    return PDFB_OK;
}

extern "C" int pdfb_lhagrid_get_xs(const pdfb_lhagrid *g, int *x_offsets, double *x_knots, int *q_offsets, double *q_knots,
                                   int *pids, double *values)
{
    if (!g || !x_offsets || !x_knots || !q_offsets || !q_knots || !pids || !values) return PDFB_EINVAL;
    memcpy(x_offsets, g->x_off.data(), sizeof(int) * g->x_off.size());
    memcpy(x_knots, g->x.data(), sizeof(double) * g->x.size());
    memcpy(q_offsets, g->q_off.data(), sizeof(int) * g->q_off.size());
    memcpy(q_knots, g->q.data(), sizeof(double) * g->q.size());
    memcpy(pids, g->pids.data(), sizeof(int) * g->pids.size());
    memcpy(values, g->values.data(), sizeof(double) * g->values.size());
    return PDFB_OK;
}

extern "C" void pdfb_lhagrid_free(pdfb_lhagrid *g) { delete g; }

// "Key: [a, b, ...]" of a metadata file; the list may continue over several lines
static int read_list(const std::string &s, const char *key, std::vector<double> &out)
{
    out.clear();
    const std::string k = std::string(key) + ":";
    size_t p = 0;
    for (;;) {  // the key at the start of a line
        p = s.find(k, p);
        if (p == std::string::npos) return PDFB_EFORMAT;
        if (p == 0 || s[p - 1] == '\n') break;
        p += k.size();
    }
    size_t a = s.find('[', p), line_end = s.find('\n', p);
    if (a == std::string::npos || (line_end != std::string::npos && a > line_end)) return PDFB_EFORMAT;
    size_t b = s.find(']', a);
    if (b == std::string::npos) return PDFB_EFORMAT;
    std::string body = s.substr(a + 1, b - a - 1);
    for (char &c : body) if (c == '\n' || c == '\r') c = ' ';
    return parse_doubles(body.data(), body.data() + body.size(), out) ? PDFB_OK : PDFB_EFORMAT;
}

// alpha_s nodes of a metadata file: AlphaS_Qs (GeV; a repeated Q marks a threshold) and AlphaS_Vals.
// *n receives the node count; if cap >= count the arrays are filled, else only *n is set (query).
extern "C" int pdfb_lhapdf_info_alphas(const char *info_path, int cap, double *q_knots, double *alphas, int *n)
{
    if (!info_path || !n) return PDFB_EINVAL;
    *n = 0;
    std::string s;
    if (!read_all(info_path, s)) return PDFB_EIO;
    std::vector<double> q, a;
    int rc = read_list(s, "AlphaS_Qs", q);
    if (!rc) rc = read_list(s, "AlphaS_Vals", a);
    if (rc) return rc;
    if (q.size() != a.size() || q.size() < 2) return PDFB_EFORMAT;
    *n = (int)q.size();
    if (cap >= *n) {
        if (!q_knots || !alphas) return PDFB_EINVAL;
        memcpy(q_knots, q.data(), sizeof(double) * q.size());
        memcpy(alphas, a.data(), sizeof(double) * a.size());
    }
    return PDFB_OK;
}

// NumMembers of a metadata file (1 if the key is absent)
extern "C" int pdfb_lhapdf_info_members(const char *info_path, int *n_members)
{
    if (!info_path || !n_members) return PDFB_EINVAL;
    *n_members = 1;
    std::string s;
    if (!read_all(info_path, s)) return PDFB_EIO;
    size_t p = s.find("NumMembers:");
    if (p != std::string::npos && (p == 0 || s[p - 1] == '\n')) {
        int v = atoi(s.c_str() + p + 11);
        if (v < 1) return PDFB_EFORMAT;
        *n_members = v;
    }
    return PDFB_OK;
}
