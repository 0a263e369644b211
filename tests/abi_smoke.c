/* C99 caller of the C ABI (include/dedisp.h): proves the header compiles as plain C and that the
 * host-only entry points work without a device.  Built and run by tests/test_abi_host.py:
 *     gcc -std=c99 -Wall -Werror -Iinclude tests/abi_smoke.c -o abi_smoke <libdedisp_b200.so>
 * Checks the eq. 1 hand values of SURVEY.md section 8c P1: 128 channels from 150 MHz
 * down in 0.05 MHz steps, t_samp 0.1 ms: channel 127 at DM 3.0 -> 500 samples, at DM 6.3 -> 1050. */
#include <stdio.h>
#include <stdlib.h>

#include "dedisp.h"

#define CHECK(cond) do { if (!(cond)) { fprintf(stderr, "abi_smoke: %s failed (line %d)\n", #cond, __LINE__); return 1; } } while (0)

int main(void)
{
    enum { NCH = 128, NDM = 64 };
    double dm[NDM];
    int32_t *tab;
    dedisp_plan *plan = NULL;
    dedisp_stream *stream = NULL;
    dedisp_survey *survey = NULL;
    dedisp_pass pass = {0.0, 0.1, 24, 12, 2};
    int64_t info[14], total = 0;
    int d, c;

    for (d = 0; d < NDM; ++d)
        dm[d] = d * 0.1;
    CHECK(dedisp_plan_create(&plan, NCH, 150.0, 0.05, 0.1, dm, NDM, 0, 0) == DEDISP_OK);
    CHECK(dedisp_plan_nchans(plan) == NCH && dedisp_plan_ndm(plan) == NDM && dedisp_plan_nsub(plan) == 0);
    CHECK(dedisp_plan_max_delay(plan) == 1050);
    tab = (int32_t *)malloc(sizeof(int32_t) * NCH * NDM);
    CHECK(tab != NULL);
    CHECK(dedisp_plan_get_shifts(plan, tab) == DEDISP_OK);
    CHECK(tab[30 * NCH + 127] == 500 && tab[30 * NCH + 64] == 244 && tab[63 * NCH + 127] == 1050);
    for (d = 0; d < NDM; ++d)
        CHECK(tab[d * NCH] == 0);                       /* reference = channel 0 (reading R3) */
    for (c = 0; c < NCH; ++c)
        CHECK(tab[c] == 0);                             /* DM 0 */
    CHECK(dedisp_plan_window_info(plan, info) == DEDISP_OK && info[0] == 1 && info[10] >= 1);
    CHECK(dedisp_plan_get_subband_shifts(plan, NULL, NULL, NULL, NULL) == DEDISP_ESTATE);
    /* no dedisp_plan_reserve yet: execute must refuse instead of allocating */
    CHECK(dedisp_execute(plan, tab, tab, DEDISP_F32, 16, 1072, 16, 1, NULL) == DEDISP_ESTATE);
    CHECK(dedisp_execute(plan, tab, tab, DEDISP_F32, 16, 8, 16, 1, NULL) == DEDISP_ESHAPE);
    CHECK(dedisp_stream_create(&stream, NULL, DEDISP_U8, 1024, 1) == DEDISP_EINVAL && stream == NULL);
    CHECK(dedisp_plan_destroy(plan) == DEDISP_OK);
    CHECK(dedisp_plan_create(&plan, 0, 150.0, 0.05, 0.1, dm, NDM, 0, 0) == DEDISP_EINVAL && plan == NULL);
    CHECK(dedisp_survey_create(&survey, NCH, 150.0, 0.05, 0.1, 8, &pass, 1) == DEDISP_OK);
    CHECK(dedisp_survey_npass(survey) == 1 && dedisp_survey_max_delay(survey) > 0);
    CHECK(dedisp_survey_out_layout(survey, 1000, 1, NULL, NULL, NULL, &total) == DEDISP_OK && total == 24 * 500);
    CHECK(dedisp_survey_destroy(survey) == DEDISP_OK);
    CHECK(dedisp_strerror(DEDISP_ESHAPE)[0] == 's');
    free(tab);
    printf("abi_smoke ok: %s\n", dedisp_version());
    return 0;
}
