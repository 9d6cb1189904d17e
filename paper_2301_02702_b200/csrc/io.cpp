// io.cpp -- files for the objects that cross the boundary (PAPER.md:93 Fig 1 "each arrow represents a file", :99-101):
// scanner + sequence in, raw signal out.  Host only.
//
// The paper reads Pulseq files and writes ISMRM Raw Data, but fixes nothing of either format beyond its name, and no
// sample file of either is available here; a reader written from memory of a third-party format could be pinned by
// nothing.  What is implemented is therefore this library's OWN container for exactly the arrays of bloch_sequence /
// bloch_scanner and for the raw samples -- NOT Pulseq, NOT ISMRMRD.  It is a line-oriented text
// file; every number is written as a C99 hexadecimal floating-point literal ("%a"), so a round trip is bit-exact and
// a plan built from a file has bitwise the tables of a plan built from the arrays (tests/test_host_io.py).
//
//   bloch-sequence 1
//   scanner <gamma> <B0> <G_max> <S_max>
//   t_end <t_end>
//   gradient <axis 0|1|2> <n>          followed by n lines  "<t> <G>"
//   rf <n>                             followed by n lines  "<t> <dt> <re> <im>"
//   adc <n>                            followed by n lines  "<t>"
//   end
//
//   bloch-signal 1
//   rows <n_rows> samples <n_adc>      rows = 1 (SUM_ALL), coils, spins or groups
//   times <0|1>                        1: every sample line starts with its ADC time
//   row <r>                            followed by n_adc lines  "[<t>] <re> <im>"
//   end
#include <cerrno>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "internal.h"

struct bloch_sequence_file {
    bloch_scanner scanner{};
    std::vector<double> g_t[3], g_v[3];
    std::vector<double> rf_t, rf_dt, rf_re, rf_im, adc_t;
    double t_end = 0;
};

namespace {

using bloch::fail;

struct File {
    FILE *f = nullptr;
    ~File() { if (f) std::fclose(f); }
};

// one number; strtod reads hexadecimal floating-point literals exactly
bool read_double(FILE *f, double *out) {
    char tok[128];
    if (std::fscanf(f, "%127s", tok) != 1) return false;
    char *end = nullptr;
    errno = 0;
    const double v = std::strtod(tok, &end);
    if (end == tok || *end != 0) return false;
    *out = v;
    return true;
}
bool read_count(FILE *f, long long *out) {
    return std::fscanf(f, "%lld", out) == 1 && *out >= 0 && *out <= (1ll << 40);
}

}  // namespace

extern "C" {

int bloch_sequence_write(const char *path, const bloch_scanner *scanner, const bloch_sequence *seq) {
    if (!path || !seq) return fail(BLOCH_EINVAL, "NULL path or sequence");
    for (int a = 0; a < 3; ++a)
        if (seq->g_n[a] < 0 || (seq->g_n[a] > 0 && (!seq->g_t[a] || !seq->g_v[a])))
            return fail(BLOCH_EINVAL, "gradient arrays NULL or negative count");
    if (seq->rf_n < 0 || (seq->rf_n > 0 && (!seq->rf_t || !seq->rf_dt || !seq->rf_re || !seq->rf_im)))
        return fail(BLOCH_EINVAL, "RF arrays NULL or negative count");
    if (seq->adc_n < 0 || (seq->adc_n > 0 && !seq->adc_t)) return fail(BLOCH_EINVAL, "ADC array NULL");
    File out;
    out.f = std::fopen(path, "w");
    if (!out.f) return fail(BLOCH_EINVAL, std::string("cannot open for writing: ") + path);
    FILE *f = out.f;
    const bloch_scanner sc = scanner ? *scanner : bloch_scanner{0, 0, 0, 0};
    std::fprintf(f, "bloch-sequence 1\nscanner %a %a %a %a\nt_end %a\n", sc.gamma, sc.B0, sc.G_max, sc.S_max, seq->t_end);
    for (int a = 0; a < 3; ++a) {
        std::fprintf(f, "gradient %d %lld\n", a, (long long)seq->g_n[a]);
        for (int64_t i = 0; i < seq->g_n[a]; ++i) std::fprintf(f, "%a %a\n", seq->g_t[a][i], seq->g_v[a][i]);
    }
    std::fprintf(f, "rf %lld\n", (long long)seq->rf_n);
    for (int64_t i = 0; i < seq->rf_n; ++i)
        std::fprintf(f, "%a %a %a %a\n", seq->rf_t[i], seq->rf_dt[i], seq->rf_re[i], seq->rf_im[i]);
    std::fprintf(f, "adc %lld\n", (long long)seq->adc_n);
    for (int64_t i = 0; i < seq->adc_n; ++i) std::fprintf(f, "%a\n", seq->adc_t[i]);
    std::fprintf(f, "end\n");
    if (std::ferror(f)) return fail(BLOCH_EINVAL, std::string("write error: ") + path);
    return BLOCH_OK;
}

int bloch_sequence_read(const char *path, bloch_sequence_file **out) {
    if (!path || !out) return fail(BLOCH_EINVAL, "NULL path or out");
    *out = nullptr;
    File in;
    in.f = std::fopen(path, "r");
    if (!in.f) return fail(BLOCH_EINVAL, std::string("cannot open: ") + path);
    FILE *f = in.f;
    char word[64];
    int version = 0;
    if (std::fscanf(f, "%63s %d", word, &version) != 2 || std::strcmp(word, "bloch-sequence") != 0 || version != 1)
        return fail(BLOCH_EINVAL, "not a bloch-sequence version 1 file (this is the library's own format, not Pulseq)");
    bloch_sequence_file *sf = new (std::nothrow) bloch_sequence_file();
    if (!sf) return fail(BLOCH_ENOMEM, "host allocation failed");
    bool have_scanner = false, have_end = false, ended = false;
    auto bad = [&](const char *what) {
        delete sf;
        return fail(BLOCH_EINVAL, std::string("bloch-sequence file: ") + what);
    };
    try {
        while (!ended && std::fscanf(f, "%63s", word) == 1) {
            if (!std::strcmp(word, "scanner")) {
                if (!read_double(f, &sf->scanner.gamma) || !read_double(f, &sf->scanner.B0) ||
                    !read_double(f, &sf->scanner.G_max) || !read_double(f, &sf->scanner.S_max))
                    return bad("malformed scanner line");
                have_scanner = true;
            } else if (!std::strcmp(word, "t_end")) {
                if (!read_double(f, &sf->t_end)) return bad("malformed t_end line");
                have_end = true;
            } else if (!std::strcmp(word, "gradient")) {
                int axis = -1;
                long long n = 0;
                if (std::fscanf(f, "%d", &axis) != 1 || axis < 0 || axis > 2 || !read_count(f, &n))
                    return bad("malformed gradient header");
                sf->g_t[axis].resize((size_t)n);
                sf->g_v[axis].resize((size_t)n);
                for (long long i = 0; i < n; ++i)
                    if (!read_double(f, &sf->g_t[axis][(size_t)i]) || !read_double(f, &sf->g_v[axis][(size_t)i]))
                        return bad("truncated gradient section");
            } else if (!std::strcmp(word, "rf")) {
                long long n = 0;
                if (!read_count(f, &n)) return bad("malformed rf header");
                sf->rf_t.resize((size_t)n); sf->rf_dt.resize((size_t)n); sf->rf_re.resize((size_t)n); sf->rf_im.resize((size_t)n);
                for (long long i = 0; i < n; ++i)
                    if (!read_double(f, &sf->rf_t[(size_t)i]) || !read_double(f, &sf->rf_dt[(size_t)i]) ||
                        !read_double(f, &sf->rf_re[(size_t)i]) || !read_double(f, &sf->rf_im[(size_t)i]))
                        return bad("truncated rf section");
            } else if (!std::strcmp(word, "adc")) {
                long long n = 0;
                if (!read_count(f, &n)) return bad("malformed adc header");
                sf->adc_t.resize((size_t)n);
                for (long long i = 0; i < n; ++i)
                    if (!read_double(f, &sf->adc_t[(size_t)i])) return bad("truncated adc section");
            } else if (!std::strcmp(word, "end")) {
                ended = true;
            } else {
                return bad("unknown section");
            }
        }
    } catch (const std::bad_alloc &) {
        delete sf;
        return fail(BLOCH_ENOMEM, "host allocation failed while reading the sequence file");
    }
    if (!ended || !have_scanner || !have_end) return bad("missing scanner / t_end / end");
    *out = sf;
    return BLOCH_OK;
}

int bloch_sequence_file_get(const bloch_sequence_file *file, bloch_scanner *scanner, bloch_sequence *seq) {
    if (!file || !seq) return fail(BLOCH_EINVAL, "NULL argument");
    if (scanner) *scanner = file->scanner;
    for (int a = 0; a < 3; ++a) {
        seq->g_t[a] = file->g_t[a].data();
        seq->g_v[a] = file->g_v[a].data();
        seq->g_n[a] = (int64_t)file->g_t[a].size();
    }
    seq->rf_t = file->rf_t.data(); seq->rf_dt = file->rf_dt.data();
    seq->rf_re = file->rf_re.data(); seq->rf_im = file->rf_im.data();
    seq->rf_n = (int64_t)file->rf_t.size();
    seq->adc_t = file->adc_t.data();
    seq->adc_n = (int64_t)file->adc_t.size();
    seq->t_end = file->t_end;
    return BLOCH_OK;
}

int bloch_sequence_file_free(bloch_sequence_file *file) {
    delete file;
    return BLOCH_OK;
}

int bloch_signal_write(const char *path, const float *h_signal, int64_t n_rows, int64_t n_adc, const double *h_adc_t) {
    if (!path || n_rows < 0 || n_adc < 0 || (n_rows * n_adc > 0 && !h_signal))
        return fail(BLOCH_EINVAL, "NULL path / signal or negative size");
    File out;
    out.f = std::fopen(path, "w");
    if (!out.f) return fail(BLOCH_EINVAL, std::string("cannot open for writing: ") + path);
    FILE *f = out.f;
    std::fprintf(f, "bloch-signal 1\nrows %lld samples %lld\ntimes %d\n", (long long)n_rows, (long long)n_adc, h_adc_t ? 1 : 0);
    for (int64_t r = 0; r < n_rows; ++r) {
        std::fprintf(f, "row %lld\n", (long long)r);
        const float *row = h_signal + 2 * r * n_adc;
        for (int64_t j = 0; j < n_adc; ++j) {
            if (h_adc_t) std::fprintf(f, "%a ", h_adc_t[j]);
            std::fprintf(f, "%a %a\n", (double)row[2 * j], (double)row[2 * j + 1]);
        }
    }
    std::fprintf(f, "end\n");
    if (std::ferror(f)) return fail(BLOCH_EINVAL, std::string("write error: ") + path);
    return BLOCH_OK;
}

int bloch_signal_read(const char *path, float *h_signal, int64_t capacity_complex, int64_t *n_rows, int64_t *n_adc,
                      double *h_adc_t) {
    if (!path || !n_rows || !n_adc) return fail(BLOCH_EINVAL, "NULL argument");
    File in;
    in.f = std::fopen(path, "r");
    if (!in.f) return fail(BLOCH_EINVAL, std::string("cannot open: ") + path);
    FILE *f = in.f;
    char w1[32], w2[32];
    int version = 0, times = 0;
    long long rows = 0, samples = 0;
    if (std::fscanf(f, "%31s %d", w1, &version) != 2 || std::strcmp(w1, "bloch-signal") != 0 || version != 1)
        return fail(BLOCH_EINVAL, "not a bloch-signal version 1 file (this is the library's own format, not ISMRMRD)");
    if (std::fscanf(f, "%31s %lld %31s %lld", w1, &rows, w2, &samples) != 4 || std::strcmp(w1, "rows") || std::strcmp(w2, "samples") ||
        rows < 0 || samples < 0)
        return fail(BLOCH_EINVAL, "bloch-signal file: malformed size line");
    if (std::fscanf(f, "%31s %d", w1, &times) != 2 || std::strcmp(w1, "times")) return fail(BLOCH_EINVAL, "bloch-signal file: malformed times line");
    *n_rows = rows;
    *n_adc = samples;
    if (!h_signal) return BLOCH_OK;  // size query
    if (capacity_complex < rows * samples) return fail(BLOCH_EWORKSPACE, "signal buffer too small for the file");
    for (long long r = 0; r < rows; ++r) {
        long long rr = -1;
        if (std::fscanf(f, "%31s %lld", w1, &rr) != 2 || std::strcmp(w1, "row") || rr != r)
            return fail(BLOCH_EINVAL, "bloch-signal file: malformed row header");
        for (long long j = 0; j < samples; ++j) {
            double t = 0, re = 0, im = 0;
            if (times && !read_double(f, &t)) return fail(BLOCH_EINVAL, "bloch-signal file: truncated row");
            if (!read_double(f, &re) || !read_double(f, &im)) return fail(BLOCH_EINVAL, "bloch-signal file: truncated row");
            h_signal[2 * (r * samples + j)] = (float)re;
            h_signal[2 * (r * samples + j) + 1] = (float)im;
            if (times && h_adc_t && r == 0) h_adc_t[j] = t;
        }
    }
    return BLOCH_OK;
}

}  // extern "C"
