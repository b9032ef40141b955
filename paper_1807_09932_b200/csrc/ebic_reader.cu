// ebic_reader.cu -- host side, no CUDA calls: the delimited-text matrix reader of include/ebic.h
// ("The data values might be separated by either comma, tabulator
// or semicolon. An upper left header is not required").  Product code: shares nothing with oracle/.
#include "../../include/ebic.h"

#include <cerrno>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <algorithm>
#include <atomic>
#include <new>
#include <thread>
#include <vector>

namespace {

struct Line {
    const char* begin;
    const char* end;   // one past the last character, line terminator (and a trailing '\r') excluded
};

// Splits the buffer into non-empty lines ("\n" or "\r\n"; blank lines are skipped).
std::vector<Line> split_lines(const char* buf, size_t n) {
    std::vector<Line> lines;
    const char* p = buf;
    const char* const stop = buf + n;
    while (p < stop) {
        const char* nl = static_cast<const char*>(memchr(p, '\n', static_cast<size_t>(stop - p)));
        const char* e = nl ? nl : stop;
        const char* trimmed = e;
        while (trimmed > p && (trimmed[-1] == '\r' || trimmed[-1] == ' ')) --trimmed;
        if (trimmed > p) lines.push_back({p, trimmed});
        p = nl ? nl + 1 : stop;
    }
    return lines;
}

int64_t count_fields(const Line& l, char d) {
    int64_t n = 1;
    for (const char* p = l.begin; p < l.end; ++p) n += (*p == d);
    return n;
}

char detect_delimiter(const Line& header) {
    const char cand[3] = {'\t', ';', ','};            // a tab or semicolon wins over commas inside names
    for (char c : cand)
        if (memchr(header.begin, c, static_cast<size_t>(header.end - header.begin))) return c;
    return 0;
}

// One numeric field [b, e): surrounding blanks and double quotes are ignored; empty, NA, NaN, nan, N/A, null
// -> NaN (a missing cell).  Returns false if the field is not a number.
bool parse_value(const char* b, const char* e, float* out) {
    while (b < e && (*b == ' ' || *b == '"')) ++b;
    while (e > b && (e[-1] == ' ' || e[-1] == '"')) --e;
    const size_t len = static_cast<size_t>(e - b);
    if (len == 0 || (len == 2 && !strncmp(b, "NA", 2)) || (len == 3 && (!strncmp(b, "NaN", 3) || !strncmp(b, "nan", 3) || !strncmp(b, "N/A", 3))) ||
        (len == 4 && !strncmp(b, "null", 4))) {
        *out = std::numeric_limits<float>::quiet_NaN();
        return true;
    }
    char tmp[64];
    if (len >= sizeof(tmp)) return false;
    memcpy(tmp, b, len);
    tmp[len] = 0;
    char* endp = nullptr;
    errno = 0;
    const float v = strtof(tmp, &endp);               // correctly rounded decimal -> float32 (glibc), also inf / 1e-3 / hex
    if (endp != tmp + len) return false;
    *out = v;                                          // overflow gives +-inf, underflow a denormal or 0: kept as parsed
    return true;
}

}  // namespace

extern "C" {

int ebic_read_delimited(const char* path, char delimiter, float** matrix, int64_t* rows, int32_t* cols) {
    if (matrix) *matrix = nullptr;
    if (rows) *rows = 0;
    if (cols) *cols = 0;
    if (!path || !matrix || !rows || !cols) return EBIC_ERR_ARG;
    if (delimiter != 0 && delimiter != ',' && delimiter != '\t' && delimiter != ';') return EBIC_ERR_ARG;
    FILE* f = fopen(path, "rb");
    if (!f) return EBIC_ERR_IO;
    std::vector<char> buf;
    {
        bool bad = fseek(f, 0, SEEK_END) != 0;
        const long size = bad ? -1 : ftell(f);
        bad = bad || size < 0 || fseek(f, 0, SEEK_SET) != 0;
        if (!bad) {
            try {
                buf.resize(static_cast<size_t>(size));
            } catch (const std::bad_alloc&) {
                fclose(f);
                return EBIC_ERR_OOM;
            }
            bad = size > 0 && fread(buf.data(), 1, buf.size(), f) != buf.size();
        }
        fclose(f);
        if (bad) return EBIC_ERR_IO;
    }
    std::vector<Line> lines;
    try {
        lines = split_lines(buf.data(), buf.size());
    } catch (const std::bad_alloc&) {
        return EBIC_ERR_OOM;
    }
    if (lines.size() < 2) return EBIC_ERR_IO;          // a header line and at least one data line
    const char d = delimiter ? delimiter : detect_delimiter(lines[0]);
    if (d == 0) return EBIC_ERR_IO;
    const int64_t header_fields = count_fields(lines[0], d);
    const int64_t data_fields = count_fields(lines[1], d);
    // header = [corner,] name_1 .. name_C ; data line = row name, v_1 .. v_C
    if (header_fields != data_fields && header_fields != data_fields - 1) return EBIC_ERR_IO;
    const int64_t C = data_fields - 1, R = static_cast<int64_t>(lines.size()) - 1;
    if (C < 1 || C > 2147483647ll || R > 2147483647ll) return EBIC_ERR_IO;
    float* M = static_cast<float*>(malloc(static_cast<size_t>(R) * static_cast<size_t>(C) * sizeof(float)));
    if (!M) return EBIC_ERR_OOM;
    // rows are independent: contiguous row ranges are parsed by up to 16 host threads
    std::atomic<bool> failed(false);
    auto parse_rows = [&](int64_t r_begin, int64_t r_end) {
        for (int64_t r = r_begin; r < r_end && !failed.load(std::memory_order_relaxed); ++r) {
            const Line& l = lines[static_cast<size_t>(r) + 1];
            const char* p = static_cast<const char*>(memchr(l.begin, d, static_cast<size_t>(l.end - l.begin)));   // skip the row name
            int64_t c = 0;
            bool ok = true;
            while (p && ok) {
                const char* b = p + 1;
                const char* nx = static_cast<const char*>(memchr(b, d, static_cast<size_t>(l.end - b)));
                const char* e = nx ? nx : l.end;
                ok = c < C && parse_value(b, e, &M[r * C + c]);
                ++c;
                p = nx;
            }
            if (!ok || c != C) failed.store(true, std::memory_order_relaxed);   // not a number, or a ragged line
        }
    };
    const unsigned hw = std::thread::hardware_concurrency();
    const int64_t n_threads = std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(hw ? hw : 1, 16), R * C / 65536));
    if (n_threads == 1) {
        parse_rows(0, R);
    } else {
        std::vector<std::thread> pool;
        try {
            for (int64_t t = 0; t < n_threads; ++t) pool.emplace_back(parse_rows, R * t / n_threads, R * (t + 1) / n_threads);
        } catch (...) {                                // could not start a thread: finish what is left here
            const int64_t started = static_cast<int64_t>(pool.size());
            parse_rows(R * started / n_threads, R);
        }
        for (auto& th : pool) th.join();
    }
    if (failed.load()) {
        free(M);
        return EBIC_ERR_IO;
    }
    *matrix = M;
    *rows = R;
    *cols = static_cast<int32_t>(C);
    return EBIC_OK;
}

void ebic_free_host(void* p) { free(p); }

}  // extern "C"
